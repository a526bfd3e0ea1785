"""B200-native exact sequential Metropolis sweeps for Coulomb many-body systems (arXiv 1602.05716).

The product is ``libmcb200.so`` (CUDA sm_100a, C ABI in ``include/mcb200.h``); ``binding`` is the thin
ctypes layer over it and ``workloads`` the seeded synthetic input generator.  Importing this package does
not load the library; the first call into ``binding`` does, and raises if it is missing (no CPU fallback).
"""
__all__ = ["binding", "workloads", "build"]
