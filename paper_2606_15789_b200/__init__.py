"""anslin — B200-native tile-level rANS weight decompression fused into tcgen05 GEMM.

Product package: csrc/ (CUDA kernels + host encoder behind the C ABI of include/anslin.h) and a
thin ctypes binding (binding.py).  inputs.py holds the seeded synthetic input generators only.
"""
