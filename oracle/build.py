"""Compile the fp64 CPU oracle (test infrastructure) with gcc into oracle/libxrdvi_oracle.so.

Run as ``python oracle/build.py``; also called by ``__graft_entry__.build()``.
Building the checker is not using it: the product never loads this library.
"""
from __future__ import annotations

import pathlib
import subprocess

HERE = pathlib.Path(__file__).resolve().parent
SRC = HERE / "xrdvi_oracle.c"
LIB = HERE / "libxrdvi_oracle.so"


def build(force: bool = False) -> pathlib.Path:
    if not force and LIB.exists() and LIB.stat().st_mtime >= SRC.stat().st_mtime:
        return LIB
    cmd = ["gcc", "-O2", "-std=c11", "-fPIC", "-shared", "-fopenmp", "-ffp-contract=off",
           "-D_GNU_SOURCE", "-o", str(LIB), str(SRC), "-lm"]
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
