"""Build the product library: paper_1807_08116_b200/libsph_b200.so (sm_100a only).

nvcc -gencode arch=compute_100a,code=sm_100a -lineinfo -O3, no --use_fast_math (the cell-key and
cutoff code paths are bit-exact FP32 sequences).  Cross-compiles without a GPU.
"""
from __future__ import annotations

import fcntl
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
PKG = os.path.dirname(HERE)
LIB = os.path.join(PKG, "libsph_b200.so")
SOURCES = ["api.cu", "gravity.cu", "gravity_sym.cu", "grid.cu", "sph.cu", "sph_dense.cu", "sph_dense_rho.cu", "step.cu", "host.cu", "nbrlist.cu", "noalloc.cu"]
DEPS = SOURCES + ["common.cuh", "grav_dev.cuh", "sph_dev.cuh", "sph_dense_dev.cuh", "tma_dev.cuh", os.path.join("..", "..", "include", "sph_b200.h")]


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(os.path.join(HERE, d)) > t for d in DEPS)


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile if stale.  Safe when several processes call it at once (torchrun ranks on a fresh checkout): one holds an
    exclusive lock on libsph_b200.so.lock and compiles into its OWN temporary name before the atomic rename; the others
    wait on the lock and then find the library fresh."""
    if not force and not _stale():
        return LIB
    with open(LIB + ".lock", "w") as lock:
        fcntl.flock(lock, fcntl.LOCK_EX)
        try:
            if not force and not _stale():          # another process built it while this one waited
                return LIB
            nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
            tmp = f"{LIB}.{os.getpid()}.tmp"
            cmd = [nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
                   "-Xcompiler", "-fPIC", "-shared", "-o", tmp]
            if verbose:
                cmd += ["-Xptxas", "-v"]
            cmd += [os.path.join(HERE, s) for s in SOURCES]
            try:
                subprocess.run(cmd, check=True)
                os.replace(tmp, LIB)
            finally:
                if os.path.exists(tmp):
                    os.unlink(tmp)
        finally:
            fcntl.flock(lock, fcntl.LOCK_UN)
    return LIB


if __name__ == "__main__":
    import sys
    print(build(force=True, verbose="-v" in sys.argv))
