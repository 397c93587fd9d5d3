"""CPU-side checks of the boundary and the host logic (no GPU, no compute calls): the C-ABI library
builds for sm_100a, loads, and exports every symbol include/hard.h declares; the binding fails loudly
without a device; bench.py's rank aggregation works over gloo with world_size 2."""
import os
import re
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_symbols():
    src = open(os.path.join(ROOT, "include", "hard.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(hard_[a-z0-9_]+)\s*\(", src)))


def test_library_builds_and_exports_every_declared_symbol():
    from paper_2509_08971_b200 import build, hard
    build.build()
    L = hard.lib()
    decl = _declared_symbols()
    assert len(decl) >= 18 and "hard_create" in decl and "hard_step" in decl
    for name in decl:
        assert hasattr(L, name), "libhard_b200.so does not export %s" % name
    assert sorted(hard.EXPORTS) == decl
    # the dynamic symbol table agrees (no C++ mangling on the boundary)
    out = subprocess.run(["nm", "-D", "--defined-only", hard.LIB_PATH], capture_output=True, text=True).stdout
    for name in decl:
        assert re.search(r"\sT\s+%s$" % name, out, flags=re.M), name
    # the fp64-peak probe is a separate library with its own header: not part of the product ABI
    assert "hard_probe_fp64_peak" not in out
    pout = subprocess.run(["nm", "-D", "--defined-only", hard.PROBE_LIB_PATH], capture_output=True, text=True).stdout
    assert re.search(r"\sT\s+hard_probe_fp64_peak$", pout, flags=re.M)
    assert "hard_probe_fp64_peak" in open(os.path.join(ROOT, "include", "hard_probe.h")).read()


def build_cabi_program():
    """gcc tests/test_cabi.c -I include against libhard_b200.so -> tests/test_cabi (plain C, no Python in the loop)."""
    from paper_2509_08971_b200 import build, hard
    build.build()
    exe = os.path.join(ROOT, "tests", "test_cabi.bin")
    libdir = os.path.dirname(hard.LIB_PATH)
    cmd = ["gcc", "-std=c99", "-Wall", "-Werror", "-O1", "-I", os.path.join(ROOT, "include"),
           os.path.join(ROOT, "tests", "test_cabi.c"), "-o", exe, "-L", libdir, "-lhard_b200",
           "-Wl,-rpath," + libdir, "-lm"]
    subprocess.check_call(cmd)
    return exe


def test_c_program_compiles_against_the_header():
    # the boundary is a C ABI — a C99 compiler accepts include/hard.h as it stands and the five
    # north-star calls link; the program itself runs on the GPU box (tests/test_gpu_api.py::test_cabi_c_program)
    exe = build_cabi_program()
    assert os.path.exists(exe)
    syms = subprocess.run(["nm", "-D", "--undefined-only", exe], capture_output=True, text=True).stdout
    for name in ("hard_create", "hard_set_state", "hard_step", "hard_get_state", "hard_max_dt"):
        assert name in syms


def test_sass_contains_tma_and_fp64_pipe_instructions():
    from paper_2509_08971_b200 import build, hard
    build.build()
    sass = subprocess.run(["cuobjdump", "-sass", hard.LIB_PATH], capture_output=True, text=True).stdout
    assert "UTMALDG" in sass            # cp.async.bulk.tensor (TMA) in the stage kernel
    assert "SYNCS" in sass              # mbarrier
    assert "DFMA" in sass and "SHFL" in sass
    assert "sm_100a" in subprocess.run(["cuobjdump", "-lelf", hard.LIB_PATH], capture_output=True, text=True).stdout


def test_no_cpu_fallback():
    import torch
    from paper_2509_08971_b200 import hard
    if torch.cuda.is_available():
        pytest.skip("needs a box without a GPU")
    with pytest.raises(hard.HardError) as e:
        hard.Hard(16, 16, 16, 1.4, 0, torch_workspace=False)
    assert "no CPU fallback" in str(e.value)
    # argument errors are reported before any device is touched
    with pytest.raises(hard.HardError):
        hard.Hard(0, 1, 1, 1.4, 0, torch_workspace=False)


def test_oracle_is_not_imported_by_the_product():
    pkg = os.path.join(ROOT, "paper_2509_08971_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt and "hard_oracle" not in txt, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".cpp")):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert not re.search(r"^\s*(import|from)\s+paper_2509_08971_b200", txt, flags=re.M), f
            assert "#include \"../paper" not in txt and "hard_device.cuh" not in txt and "hard_kernels.cuh" not in txt, f


_WORKER = r"""
import os, sys
sys.path.insert(0, %r)
import torch.distributed as dist
import bench
dist.init_process_group("gloo", init_method="tcp://127.0.0.1:%%s" %% sys.argv[2], rank=int(sys.argv[1]), world_size=2)
rank = dist.get_rank()
ms = bench.max_over_ranks(100.0 + 50.0 * rank)
assert ms == 150.0, ms
v = bench.job_throughput(1000, 2, 10, ms, dist.get_world_size())
assert abs(v - 2 * 1000 * 2 * 10 / 0.150) < 1e-6, v
dist.barrier()
dist.destroy_process_group()
print("ok", rank)
"""


def test_rank_aggregation_gloo_world_size_2(tmp_path):
    import socket
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    script = tmp_path / "worker.py"
    script.write_text(_WORKER % ROOT)
    procs = [subprocess.Popen([sys.executable, str(script), str(r), str(port)], stdout=subprocess.PIPE,
                              stderr=subprocess.STDOUT, text=True) for r in range(2)]
    outs = [p.communicate(timeout=300)[0] for p in procs]
    for r, (p, o) in enumerate(zip(procs, outs)):
        assert p.returncode == 0 and ("ok %d" % r) in o, o


def test_reference_arm_prints_contract_line():
    import json
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "1",
                          "--warmup", "0"], capture_output=True, text=True, timeout=600)
    assert out.returncode == 0, out.stderr
    line = json.loads(out.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["cpu_baseline"]["kind"] == "oracle" and line["value"] > 0
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["unit"] == "cell-stage-updates/s"


def test_noalloc_entry_point_checks_arguments_before_touching_a_device():
    """hard_max_dt_noalloc (include/hard.h): size and null checks come first and need no GPU; on a box without one a
    well-formed call fails loudly with HARD_ERR_CUDA (no CPU fallback), it does not compute anything on the host."""
    import ctypes
    import torch
    from paper_2509_08971_b200 import hard
    L = hard.lib()
    buf = (ctypes.c_double * 8)()
    p = ctypes.addressof(buf)
    err = lambda: L.hard_noalloc_last_error().decode()
    assert L.hard_max_dt_noalloc(0, 1, 1, 1.4, 1.0, 1.0, 1.0, p, p, p, p, p, p, None) == hard.ERR_ARG
    assert L.hard_max_dt_noalloc(8, 1, 1, 1.0, 1.0, 1.0, 1.0, p, p, p, p, p, p, None) == hard.ERR_ARG          # gamma <= 1
    assert L.hard_max_dt_noalloc(8, 1, 1, 1.4, 0.0, 1.0, 1.0, p, p, p, p, p, p, None) == hard.ERR_ARG          # dx <= 0
    assert L.hard_max_dt_noalloc(1, 1, 1, 1.4, 1.0, 1.0, 1.0, p, p, p, p, p, p, None) == hard.ERR_ARG          # no active direction
    assert L.hard_max_dt_noalloc(8, 1, 1, 1.4, 1.0, 1.0, 1.0, p, p, None, p, p, p, None) == hard.ERR_ARG and "null" in err()
    assert L.hard_max_dt_noalloc(4096, 4096, 3, 1.4, 1.0, 1.0, 1.0, p, p, p, p, p, p, None) == hard.ERR_ARG    # 50 331 648 cells
    assert "HARD_NOALLOC_MAX_CELLS" in err() and str(hard.NOALLOC_MAX_CELLS) in err()
    assert hard.NOALLOC_MAX_CELLS == 1 << 25
    hdr = open(os.path.join(ROOT, "include", "hard.h")).read()
    assert "#define HARD_NOALLOC_MAX_CELLS (1LL << 25)" in hdr
    if not torch.cuda.is_available():
        rc = L.hard_max_dt_noalloc(8, 1, 1, 1.4, 1.0, 1.0, 1.0, p, p, p, p, p, p, None)
        assert rc == hard.ERR_CUDA and "no CPU fallback" in err()
    # the static scratch is in the library image: a 33 024-byte object in its device code, no allocation call in the source
    src = open(os.path.join(ROOT, "paper_2509_08971_b200", "csrc", "hard_noalloc.cu")).read()
    code = re.sub(r"//.*", "", src)
    assert "cudaMalloc" not in code and "cudaFree" not in code and "cudaGetSymbolAddress" in code
