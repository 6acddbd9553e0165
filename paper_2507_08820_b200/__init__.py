"""paper_2507_08820_b200 — B200-native D3Q27 regularized fluctuating lattice Boltzmann (Reg-FLBM).

The product is the C-ABI library built from csrc/ (include/rflbm.h); `binding` is a thin ctypes
layer with the same names.  Nothing is loaded at import time; the first use of the binding loads
csrc/librflbm.so and fails loudly if it is missing (there is no CPU fallback).
"""
__all__ = ["binding", "synthetic", "build"]
