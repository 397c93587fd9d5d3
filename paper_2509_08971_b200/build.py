"""Build libhard_b200.so (the C-ABI of include/hard.h) and libhard_probe.so (the fp64-peak probe of
include/hard_probe.h) in-tree with nvcc for sm_100a (cross-compiles without a GPU)."""
from __future__ import annotations

import os
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
INC = os.path.join(_HERE, "..", "include")
LIB = os.path.join(_HERE, "libhard_b200.so")
PROBE_LIB = os.path.join(_HERE, "libhard_probe.so")
TARGETS = {
    LIB: (["hard_api.cu", "hard_noalloc.cu"], ["hard_api.cu", "hard_noalloc.cu", "hard_kernels.cuh", "hard_stage3d.cuh",
                                               "hard_device.cuh", os.path.join(INC, "hard.h")]),
    PROBE_LIB: (["hard_probe.cu"], ["hard_probe.cu", os.path.join(INC, "hard_probe.h")]),
}
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-Xcompiler", "-fPIC", "-shared"]


def _nvcc():
    for p in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if p and (os.path.isabs(p) and os.path.exists(p) or not os.path.isabs(p)):
            return p
    return "nvcc"


def build(force: bool = False, verbose: bool = False) -> str:
    for lib, (sources, deps) in TARGETS.items():
        newest = max(os.path.getmtime(os.path.join(CSRC, d)) for d in deps)
        if not force and os.path.exists(lib) and os.path.getmtime(lib) >= newest:
            continue
        tmp = lib + ".tmp.%d" % os.getpid()
        cmd = [_nvcc(), *NVCC_FLAGS, *(["-Xptxas", "-v"] if verbose else []),
               *[os.path.join(CSRC, s) for s in sources], "-o", tmp]
        subprocess.check_call(cmd)
        os.replace(tmp, lib)
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose=True))
