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
SRC = [os.path.join(HERE, "csrc", f) for f in ("prepare.cu", "solve.cu", "mg.cu", "noalloc.cu")]
DEPS = ([os.path.join(HERE, "csrc", f) for f in sorted(os.listdir(os.path.join(HERE, "csrc")))]
        + [os.path.join(ROOT, "include", "implicit_filter.h")])
LIB = os.path.join(HERE, "libimplicit_filter.so")

NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC", "-I", os.path.join(ROOT, "include")]
OBJ_DIR = os.path.join(HERE, "build")


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(d) > t for d in DEPS)


def build(force: bool = False, verbose: bool = False) -> str:
    """One nvcc per translation unit, side by side, then the link (the three files take about a minute in a row)."""
    if force or needs_build():
        nvcc = os.environ.get("NVCC", "nvcc")
        extra = os.environ.get("IF_NVCC_EXTRA", "").split()      # e.g. -DIF_TILE_ROWS=64 (tuning experiments)
        os.makedirs(OBJ_DIR, exist_ok=True)
        objs, procs = [], []
        for src in SRC:
            obj = os.path.join(OBJ_DIR, os.path.basename(src) + ".o")
            objs.append(obj)
            cmd = [nvcc] + NVCC_FLAGS + extra + (["-Xptxas", "-v"] if verbose else []) + ["-c", "-o", obj, src]
            procs.append((cmd, subprocess.Popen(cmd)))
        for cmd, p in procs:
            if p.wait() != 0:
                raise subprocess.CalledProcessError(p.returncode, cmd)
        subprocess.run([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-o", LIB] + objs, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
