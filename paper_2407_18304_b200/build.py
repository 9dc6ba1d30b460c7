"""Build libmgrhd.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a.

    python -m paper_2407_18304_b200.build [--force] [--check]

nvcc cross-compiles without a GPU.  The .so is git-ignored but travels to the GPU box.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libmgrhd.so")
SOURCES = ["mgrhd_api.cu"]
DEPS = ["mgrhd_api.cu", "mgrhd_kernels.cuh", "mgrhd_general.cuh", "mgrhd_transport.cuh", "mgrhd_planck.cuh", "mgrhd_params.h",
        os.path.join("..", "..", "include", "mgrhd.h")]

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-O3", "-lineinfo", "-std=c++17",
    "--fmad=true",               # FMA contraction is part of the product's arithmetic
    "-Xcompiler", "-fPIC", "-shared",
]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.sep not in cand or os.path.exists(cand)):
            return cand
    raise RuntimeError("nvcc not found")


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(os.path.join(CSRC, d)) > t for d in DEPS)


def build(force: bool = False, verbose: bool = False, check: bool = False) -> str:
    """check=True: the bounds-checked debug build (the update kernel's dynamic shared-memory, state and
    scratch indices are tested where they are used; a violation traps; see DESIGN.md section 11 for what
    is not covered).  Always rebuild without it before timing anything."""
    if force or check or needs_build():
        cmd = ([_nvcc()] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else [])
               + (["-DMGRHD_BOUNDS_CHECK"] if check else []) + ["-o", LIB] + SOURCES)
        subprocess.run(cmd, check=True, cwd=CSRC)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv, check="--check" in sys.argv))
