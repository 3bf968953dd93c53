"""Builds the CUDA engine in-tree: paper_1503_01722_b200/libmc_b200.so (sm_100a only).

    python -m paper_1503_01722_b200.build [--force] [--verbose]

nvcc cross-compiles without a GPU.  -fmad is left on: the fp32 arithmetic contract (R20) is
written with explicit round-to-nearest intrinsics, which nvcc never contracts.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libmc_b200.so")
SRC = [os.path.join(CSRC, "mc_engine.cu"), os.path.join(CSRC, "mc_noalloc.cu"), os.path.join(CSRC, "mc_tables.cpp"), os.path.join(CSRC, "mc_gs.cpp")]
DEPS = SRC + [os.path.join(CSRC, f) for f in ("mc_device.cuh", "mc_kernels.cuh", "mc_tables.h", "mc_gs.h")] + \
    [os.path.join(os.path.dirname(HERE), "include", "mc.h")]
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")


def build(force=False, verbose=False):
    if not force and os.path.exists(LIB) and all(os.path.getmtime(LIB) >= os.path.getmtime(s) for s in DEPS):
        return LIB
    cmd = [NVCC, "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-std=c++17", "-lineinfo",
           "-prec-div=false", "-prec-sqrt=false", "-Xcompiler", "-fPIC,-O2,-Wall,-pthread", "-shared", "-cudart", "shared", "-o", LIB] + SRC
    if verbose:
        cmd[1:1] = ["-Xptxas", "-v"]
    subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
