"""Build step of the package: compiles csrc/beagle.cu into libbeagle_b200.so (in-tree, sm_100a only).

nvcc cross-compiles without a GPU. The output sits beside this file so that it travels with the
source tree; it is git-ignored (history stays source-only).
"""
from __future__ import annotations

import os
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
SRC_DIR = os.path.join(_HERE, "csrc")
LIB = os.path.join(_HERE, "libbeagle_b200.so")
SOURCES = ["beagle.cu"]
DEPS = sorted(f for f in os.listdir(SRC_DIR) if f.endswith((".cu", ".cuh", ".inc"))) + [os.path.join("..", "..", "include", "beagle.h")]

NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-Xcompiler", "-fPIC", "-shared", "--fmad=false"]


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(os.path.join(SRC_DIR, d)) > t for d in DEPS)


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile the CUDA library if it is missing or older than its sources. Returns its path."""
    if force or _stale():
        nvcc = os.environ.get("NVCC", "nvcc")
        cmd = [nvcc, *NVCC_FLAGS, *(["-Xptxas", "-v"] if verbose else []), "-o", LIB,
               *[os.path.join(SRC_DIR, s) for s in SOURCES]]
        subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose=True))
