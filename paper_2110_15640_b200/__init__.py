"""gcmcrt-b200: B200-native (sm_100a) Monte Carlo photon-packet transport with peel-off
(next-event estimation) for albedo and emission spectra, after gCMCRT (arXiv 2110.15640).

The product is the C-ABI library `libgcmcrt.so` (include/gcmcrt.h, csrc/) and the thin
ctypes binding in `binding.py`.  Importing the package does not load the library; the
first call does, and fails loudly if it has not been built (there is no CPU fallback).
"""
__all__ = ["workloads", "binding"]
