"""kara-b200: B200-native (sm_100a) Kara sliding-window KV-cache compression step.

The product is the C-ABI library `libkara.so` (include/kara.h, csrc/); `kara` below is the thin
ctypes binding with the same entry-point names.  `inputs` holds the seeded synthetic workload
generators shared by the tests of the CUDA path and of the CPU oracle.  Importing the package
does not load the library; the first call through `paper_2607_01237_b200.kara` does, and fails
loudly if it is missing (there is no CPU fallback).
"""
__all__ = ["inputs", "kara"]
