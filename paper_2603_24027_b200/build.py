"""Build libfdtd_b200.so (the C-ABI library of include/fdtd.h) in-tree with nvcc for sm_100a.

-fmad=false: no implicit FMA contraction; every fused multiply-add in the kernels is an explicit fmaf, so the
f32 operation order is the canonical one of DESIGN.md R3.  No -use_fast_math, no FTZ, IEEE division.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libfdtd_b200.so")
SOURCES = [os.path.join(CSRC, "fdtd_api.cu")]
DEPS = SOURCES + [os.path.join(CSRC, f) for f in ("fdtd_dev.cuh", "fdtd_stencil.cuh", "fdtd_store.cuh", "fdtd_fused.cuh")] + [
    os.path.join(os.path.dirname(HERE), "include", f) for f in ("fdtd.h", "fdtd_bench.h")]
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-std=c++17", "-O3", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-fmad=false",
         "-Xcompiler", "-fPIC", "-shared", "-cudart", "static"]


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and os.path.exists(LIB) and all(os.path.getmtime(LIB) >= os.path.getmtime(d) for d in DEPS):
        return LIB
    cmd = [NVCC] + FLAGS + (["-Xptxas", "-v"] if verbose else []) + SOURCES + ["-o", LIB]
    subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
