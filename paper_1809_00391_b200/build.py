"""Builds the CUDA library (csrc/libmbt.so) in-tree with nvcc for sm_100a.

    python -m paper_1809_00391_b200.build [--force]

nvcc cross-compiles without a GPU.  Flags: -O3, -lineinfo (ncu source view), --fmad=false (every FMA in
the kernels is written out explicitly).
"""
from __future__ import annotations

import os
import shutil
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(CSRC, "libmbt.so")
SOURCES = ["mbt.cu"]
DEPS = ["mbt.cu", "mbt_kernels.cuh", "mbt_trans.cuh", "mbt_resident.cuh", "mbt_math.cuh", "mbt_coeffs.inc", "gen_coeffs.py",
        os.path.join("..", "..", "include", "mbt.h"), os.path.join("..", "build.py")]

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-O3", "-lineinfo", "--fmad=false", "-std=c++17",
    "-Xcompiler", "-fPIC,-O2,-Wall",
    "--shared",
]


def nvcc_path() -> str:
    return shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"


def up_to_date() -> bool:
    if not os.path.exists(LIB):
        return False
    t = os.path.getmtime(LIB)
    return all(os.path.getmtime(os.path.join(CSRC, d)) <= t for d in DEPS)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and up_to_date():
        return LIB
    cmd = [nvcc_path()] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-o", LIB + ".tmp"] + SOURCES
    r = subprocess.run(cmd, cwd=CSRC, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError("nvcc failed:\n" + " ".join(cmd) + "\n" + r.stdout + r.stderr)
    if verbose:
        print(r.stdout + r.stderr)
    os.replace(LIB + ".tmp", LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
