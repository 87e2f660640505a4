"""Build the product library: paper_1807_08116_b200/libsph_b200.so (sm_100a only).

nvcc -gencode arch=compute_100a,code=sm_100a -lineinfo -O3, no --use_fast_math (the cell-key and
cutoff code paths are bit-exact FP32 sequences).  Cross-compiles without a GPU.
"""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
PKG = os.path.dirname(HERE)
LIB = os.path.join(PKG, "libsph_b200.so")
SOURCES = ["api.cu", "gravity.cu", "gravity_sym.cu", "grid.cu", "sph.cu", "step.cu", "host.cu", "nbrlist.cu"]
DEPS = SOURCES + ["common.cuh", "grav_dev.cuh", os.path.join("..", "..", "include", "sph_b200.h")]


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(os.path.join(HERE, d)) > t for d in DEPS)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not _stale():
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    cmd = [nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
           "-Xcompiler", "-fPIC", "-shared", "-o", LIB + ".tmp"]
    if verbose:
        cmd += ["-Xptxas", "-v"]
    cmd += [os.path.join(HERE, s) for s in SOURCES]
    subprocess.run(cmd, check=True)
    os.replace(LIB + ".tmp", LIB)
    return LIB


if __name__ == "__main__":
    import sys
    print(build(force=True, verbose="-v" in sys.argv))
