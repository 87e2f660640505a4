"""Compile the oracle's C (test infrastructure) into oracle/libsph_oracle.so.

Flags: -O2 -fopenmp -ffp-contract=off (each FP32 line of the key / predicate code is one
IEEE operation; no -march=native so the library runs on any x86-64 host; no -ffast-math).
"""
from __future__ import annotations

import fcntl
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "sph_oracle.c")
LIB = os.path.join(HERE, "libsph_oracle.so")


def _fresh() -> bool:
    return os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(SRC)


def build(force: bool = False) -> str:
    """Compile if stale; concurrent callers serialise on a lock file and each compiles into its own temporary name."""
    if not force and _fresh():
        return LIB
    with open(LIB + ".lock", "w") as lock:
        fcntl.flock(lock, fcntl.LOCK_EX)
        try:
            if not force and _fresh():
                return LIB
            tmp = f"{LIB}.{os.getpid()}.tmp"
            cmd = ["gcc", "-O2", "-fopenmp", "-ffp-contract=off", "-fno-fast-math", "-shared", "-fPIC",
                   "-o", tmp, SRC, "-lm"]
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
    print(build(force=True))
