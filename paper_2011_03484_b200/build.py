"""Builds libglisse.so (the C-ABI library of include/glisse.h) in-tree with nvcc for sm_100a.

    python -m paper_2011_03484_b200.build [--force]

nvcc cross-compiles without a GPU.  The shared object is git-ignored but travels to the GPU box
with the repo snapshot.
"""
from __future__ import annotations

import os
import shutil
import subprocess
import sys

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
LIB = os.path.join(_HERE, "libglisse.so")
SOURCES = ["api.cu", "particles.cu", "planets.cu", "compact.cu", "snapshot.cu", "probe.cu"]
HEADERS = ["glisse_internal.cuh", "kepler.cuh", "sincos_coeffs.inc", os.path.join("..", "..", "include", "glisse.h")]

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-O3", "-std=c++17", "-lineinfo",
    "-Xcompiler", "-fPIC", "-shared",
    # the FP64 pipe is the roofline: keep fused multiply-adds, no fast-math anywhere
    "--fmad=true",
]


def nvcc() -> str:
    exe = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not os.path.exists(exe):
        raise RuntimeError("nvcc not found: the CUDA path cannot be built (there is no CPU fallback)")
    return exe


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, f) for f in SOURCES + HEADERS] + [os.path.abspath(__file__)]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile every CUDA translation unit of the library into one shared object; returns its path."""
    if force or _stale():
        tmp = LIB + f".tmp{os.getpid()}"
        cmd = [nvcc(), *NVCC_FLAGS, *(["-Xptxas", "-v"] if verbose else []),
               *[os.path.join(CSRC, f) for f in SOURCES], "-o", tmp]
        subprocess.run(cmd, check=True)
        os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
