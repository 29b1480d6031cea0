"""Build libgcmcrt.so (the C-ABI library, hand-written CUDA for sm_100a) in-tree with nvcc.

Usage: python -m paper_2110_15640_b200.build [--force] [--verbose]
nvcc cross-compiles without a GPU; the .so travels to the GPU box with the repo snapshot.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libgcmcrt.so")
SOURCES = [os.path.join(CSRC, "gcmcrt.cu")]
DEPS = SOURCES + [os.path.join(CSRC, f) for f in ("kernels.cuh", "ray.cuh", "sort.cuh", "wavefront.cuh", "device_common.cuh")] + \
    [os.path.join(os.path.dirname(HERE), "include", "gcmcrt.h")]

NVCC_FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
              "-Xcompiler", "-fPIC", "-shared", "--expt-relaxed-constexpr"]


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(f) > t for f in DEPS)


LIB_CHECKED = os.path.join(HERE, "libgcmcrt_checked.so")


def build(force: bool = False, verbose: bool = False, checked: bool = False) -> str:
    """checked = True: the variant with -DGCMCRT_CHECKED (device-side bounds and state checks, device_common.cuh) as
    libgcmcrt_checked.so; load it with GCMCRT_LIB=<path> (binding.py)."""
    lib = LIB_CHECKED if checked else LIB
    stale = not os.path.exists(lib) or any(os.path.getmtime(f) > os.path.getmtime(lib) for f in DEPS)
    if force or stale:
        nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
        tmp = lib + ".tmp.%d" % os.getpid()
        cmd = [nvcc] + NVCC_FLAGS + (["-DGCMCRT_CHECKED"] if checked else []) + (["-Xptxas", "-v"] if verbose else []) + ["-o", tmp] + SOURCES
        subprocess.run(cmd, check=True)
        os.replace(tmp, lib)
    return lib


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv, checked="--checked" in sys.argv))
