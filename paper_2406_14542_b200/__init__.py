"""B200-native nonuniform spin-0 spherical harmonic transform (nuSHT) of arXiv 2406.14542.

The product is the C-ABI library built from csrc/ (include/nusht.h); `nusht.py` is the thin
ctypes binding with the same names.  `inputs.py` holds only seeded workload generators.
Importing this package does not load the CUDA library; `paper_2406_14542_b200.nusht` does, and
raises if it has not been built (there is no CPU fallback).
"""
