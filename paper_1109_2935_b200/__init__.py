"""paper_1109_2935_b200 -- B200-native (sm_100a) Wilson-clover Dirac operator and solvers.

The product is the C-ABI library declared in include/lqcd.h (built from csrc/ into
liblqcd_b200.so); `paper_1109_2935_b200.lqcd` is the thin ctypes binding with the same
names.  Importing this package does not load the library; the first call does, and it
raises if the CUDA extension is missing (there is no CPU fallback).
"""
__all__ = ["inputs", "lqcd"]
