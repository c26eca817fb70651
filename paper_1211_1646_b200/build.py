"""Build the C-ABI CUDA library in-tree: nvcc for sm_100a only, -fmad=false (no implicit FMA contraction),
-lineinfo for ncu source pages, static cudart so the .so loads on a box without a CUDA driver.

The kernel families are separate translation units (csrc/k_*.cu, one object per precision), compiled in parallel and
linked into one shared library.  Objects go to csrc/build/ (git-ignored)."""
from __future__ import annotations

import os
import subprocess
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(CSRC, "build")
LIB = os.path.join(HERE, "libmpmc_b200.so")
# headers each source includes (directly or not)
HEADERS = {
    "mpmc.cu": ["common.cuh", "sweep.cuh", "tile.cuh", "tile4.cuh", "cluster.cuh", "aux.cuh", "kernels.h",
                os.path.join("..", "..", "include", "mpmc.h")],
    "k_general.cu": ["common.cuh", "sweep.cuh", "kernels.h"],
    "k_tile2.cu": ["common.cuh", "sweep.cuh", "tile.cuh", "kernels.h"],
    "k_tile4.cu": ["common.cuh", "sweep.cuh", "tile.cuh", "tile4.cuh", "kernels.h"],
    "k_cluster.cu": ["common.cuh", "sweep.cuh", "tile.cuh", "cluster.cuh", "kernels.h"],
}
# (source, object name, extra defines)
_PREC = [("f32", "float"), ("f64", "double")]
UNITS = [("mpmc.cu", "mpmc.o", [])] + [
    (src, f"{src[:-3]}_{sfx}.o", [f"-DMPMC_P={typ}", f"-DMPMC_SUFFIX={sfx}"])
    for src in ("k_general.cu", "k_tile2.cu", "k_tile4.cu", "k_cluster.cu") for sfx, typ in _PREC]

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-O3", "-std=c++17", "-lineinfo", "-fmad=false",
    "-Xcompiler", "-fPIC,-ffp-contract=off",
]


def _nvcc() -> str:
    return os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")


def build(force: bool = False, verbose: bool = False, extra_flags=(), lib: str = LIB) -> str:
    """Compile what is out of date and link `lib`.  extra_flags (e.g. ["-DMPMC_PHASE_CLOCKS"]) select an instrumented
    variant, which must be given its own `lib` path (its objects get their own directory)."""
    if os.environ.get("MPMC_B200_LIB") and lib == LIB:      # an explicitly chosen, already built library
        return os.environ["MPMC_B200_LIB"]
    obj_dir = OBJ if lib == LIB else OBJ + "_" + os.path.basename(lib).replace(".so", "")
    os.makedirs(obj_dir, exist_ok=True)
    stamp = os.path.join(obj_dir, "flags.txt")                # objects compiled with other flags are stale
    flags_now = " ".join(NVCC_FLAGS + list(extra_flags))
    if not os.path.exists(stamp) or open(stamp).read() != flags_now:
        force = True
        open(stamp, "w").write(flags_now)

    def compile_unit(unit):
        src, obj, defs = unit
        src_path, obj_path = os.path.join(CSRC, src), os.path.join(obj_dir, obj)
        newest = max([os.path.getmtime(os.path.join(CSRC, h)) for h in HEADERS[src]]
                     + [os.path.getmtime(src_path), os.path.getmtime(__file__)])
        if not force and os.path.exists(obj_path) and os.path.getmtime(obj_path) >= newest:
            return obj_path, False
        cmd = [_nvcc()] + NVCC_FLAGS + list(extra_flags) + defs + (["-Xptxas", "-v"] if verbose else []) + \
              ["-c", "-o", obj_path, src_path]
        subprocess.run(cmd, check=True)
        return obj_path, True

    with ThreadPoolExecutor(max_workers=min(len(UNITS), os.cpu_count() or 1)) as ex:
        results = list(ex.map(compile_unit, UNITS))
    objs = [o for o, _ in results]
    if force or any(changed for _, changed in results) or not os.path.exists(lib):
        subprocess.run([_nvcc(), "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "--cudart=static",
                        "-o", lib] + objs, check=True)
    return lib


if __name__ == "__main__":
    import sys
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
