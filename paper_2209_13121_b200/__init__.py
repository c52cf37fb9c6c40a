"""B200-native CyRSoXS forward-simulation hot path (arXiv 2209.13121).

`workloads` holds the seeded synthetic input generators; `binding` is the thin ctypes
layer over the C-ABI library `libcyrsoxs.so` declared in include/cyrsoxs.h.  Importing
the package does not load the library; `binding.load()` does and fails loudly if the
CUDA build is missing (there is no CPU fallback).
"""
__all__ = ["workloads", "binding", "build", "sharding"]
