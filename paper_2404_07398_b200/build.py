"""Builds the CUDA library in-tree: paper_2404_07398_b200/libimplicit_filter.so (sm_100a only).

    python -m paper_2404_07398_b200.build [--force]

nvcc cross-compiles without a GPU; the .so travels to the GPU box with the repository snapshot.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
SRC = [os.path.join(HERE, "csrc", f) for f in ("prepare.cu", "solve.cu", "mg.cu")]
DEPS = ([os.path.join(HERE, "csrc", f) for f in sorted(os.listdir(os.path.join(HERE, "csrc")))]
        + [os.path.join(ROOT, "include", "implicit_filter.h")])
LIB = os.path.join(HERE, "libimplicit_filter.so")

NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC", "-shared", "-I", os.path.join(ROOT, "include")]


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(d) > t for d in DEPS)


def build(force: bool = False, verbose: bool = False) -> str:
    if force or needs_build():
        nvcc = os.environ.get("NVCC", "nvcc")
        extra = os.environ.get("IF_NVCC_EXTRA", "").split()      # e.g. -DIF_TILE_ROWS=64 (tuning experiments)
        cmd = [nvcc] + NVCC_FLAGS + extra + (["-Xptxas", "-v"] if verbose else []) + ["-o", LIB] + SRC
        subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
