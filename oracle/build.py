"""Build the CPU oracle (TEST INFRASTRUCTURE) into oracle/libgcmcrt_oracle.so with gcc.

Usage: python -m oracle.build   (also called by tests/conftest.py and __graft_entry__.build()).
Building the checker is not using it: nothing in paper_2110_15640_b200/ loads this library.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "gcmcrt_oracle.c")
HDR = os.path.join(HERE, "gcmcrt_oracle.h")
LIB = os.path.join(HERE, "libgcmcrt_oracle.so")


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(f) > t for f in (SRC, HDR))


def build(force: bool = False) -> str:
    if force or needs_build():
        tmp = LIB + ".tmp.%d" % os.getpid()
        cmd = ["gcc", "-std=c99", "-O2", "-fPIC", "-shared", "-fopenmp", "-Wall", "-Wextra",
               "-D_GNU_SOURCE", "-o", tmp, SRC, "-lm"]
        subprocess.run(cmd, check=True)
        os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
