"""Compile the CUDA library (C ABI of include/xrdvi.h) for sm_100a, in-tree.

``python -m paper_2501_09308_b200.build`` or ``__graft_entry__.build()``.  nvcc cross-compiles
without a GPU; the resulting paper_2501_09308_b200/libxrdvi.so travels with the tree.
"""
from __future__ import annotations

import pathlib
import subprocess

PKG = pathlib.Path(__file__).resolve().parent
CSRC = PKG / "csrc"
LIB = PKG / "libxrdvi.so"
SOURCES = [CSRC / "xrdvi.cu"]
DEPS = SOURCES + [CSRC / "xrdvi_kernels.cuh", PKG.parent / "include" / "xrdvi.h", PKG.parent / "include" / "xrdvi_debug.h"]
MEASURE_LIB = PKG / "libxrdvi_measure.so"      # pipe-rate microbenchmark: its own library, never loaded by the product

NVCC_FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
              "-Xcompiler", "-fPIC", "-shared", "-cudart", "static"]


def build(force: bool = False, verbose: bool = False, tuning: bool = False, defines: tuple = ()) -> pathlib.Path:
    """`tuning=True` (``--tuning``) compiles with -DXRDVI_TUNING: the measurement build, in which environment knobs
    (kernel choice, chunks per warp, cost weights) steer the library for A/B runs.  The product build has none."""
    if not force and LIB.exists() and all(LIB.stat().st_mtime >= p.stat().st_mtime for p in DEPS):
        return LIB
    extra = (["-DXRDVI_TUNING"] if tuning else []) + [f"-D{d}" for d in defines]
    cmd = ["nvcc", *NVCC_FLAGS, *extra, *(["-Xptxas", "-v"] if verbose else []), "-o", str(LIB), *map(str, SOURCES)]
    subprocess.run(cmd, check=True)
    return LIB


def build_measure() -> pathlib.Path:
    """nvcc the pipe-rate microbenchmark (csrc/pipe_rates.cu, include/xrdvi_measure.h) into libxrdvi_measure.so."""
    subprocess.run(["nvcc", *NVCC_FLAGS, "-o", str(MEASURE_LIB), str(CSRC / "pipe_rates.cu")], check=True)
    return MEASURE_LIB


if __name__ == "__main__":
    import sys
    if "--measure" in sys.argv:
        print(build_measure())
    print(build(force=True, verbose="-v" in sys.argv, tuning="--tuning" in sys.argv,
                defines=tuple(a[2:] for a in sys.argv[1:] if a.startswith("-D"))))
