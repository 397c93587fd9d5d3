"""the oracle under AddressSanitizer + UndefinedBehaviorSanitizer (the GPU side has no
compute-sanitizer on this pool; the checker itself should at least be clean).  Builds oracle/hard_oracle.cpp with
tests/oracle_sanitize_driver.cpp into a stand-alone program (the sanitizer runtimes cannot be loaded into an
uninstrumented python) and runs one step per scheme x BC x {5 fields, 6 fields, 6 fields + source} on 3-D, 2-D and
1-D meshes.  Same optimisation and contraction flags as the oracle proper, so the arithmetic under test is the same."""
import os
import subprocess

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_oracle_is_clean_under_asan_and_ubsan(tmp_path):
    exe = str(tmp_path / "oracle_sanitized")
    cmd = ["g++", "-O1", "-g", "-std=c++17", "-ffp-contract=off", "-fsanitize=address,undefined",
           "-fno-sanitize-recover=all", "-fno-omit-frame-pointer", os.path.join(ROOT, "oracle", "hard_oracle.cpp"),
           os.path.join(ROOT, "tests", "oracle_sanitize_driver.cpp"), "-o", exe]
    subprocess.check_call(cmd)
    env = dict(os.environ, ASAN_OPTIONS="detect_leaks=1:abort_on_error=0", UBSAN_OPTIONS="print_stacktrace=1")
    env.pop("LD_PRELOAD", None)
    out = subprocess.run([exe], capture_output=True, text=True, env=env, timeout=600)
    assert out.returncode == 0, out.stdout + out.stderr
    assert "54 runs clean" in out.stdout
    assert "runtime error" not in out.stderr and "AddressSanitizer" not in out.stderr
