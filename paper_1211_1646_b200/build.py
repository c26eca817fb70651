"""Build the C-ABI CUDA library in-tree: nvcc for sm_100a only, -fmad=false (no implicit FMA contraction),
-lineinfo for ncu source pages, static cudart so the .so loads on a box without a CUDA driver."""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libmpmc_b200.so")
SOURCES = ["mpmc.cu"]
DEPS = ["mpmc.cu", "common.cuh", "sweep.cuh", "tile.cuh", "tile4.cuh", "aux.cuh", os.path.join("..", "..", "include", "mpmc.h")]

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-O3", "-std=c++17", "-lineinfo", "-fmad=false",
    "-Xcompiler", "-fPIC,-ffp-contract=off", "-shared", "--cudart=static",
]


def build(force: bool = False, verbose: bool = False) -> str:
    if os.environ.get("MPMC_B200_LIB"):          # an explicitly chosen, already built library (experiments)
        return os.environ["MPMC_B200_LIB"]
    newest = max(os.path.getmtime(os.path.join(CSRC, d)) for d in DEPS)
    newest = max(newest, os.path.getmtime(__file__))
    if force or not os.path.exists(LIB) or os.path.getmtime(LIB) < newest:
        nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
        cmd = [nvcc] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + \
              ["-o", LIB] + [os.path.join(CSRC, s) for s in SOURCES]
        subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    import sys
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
