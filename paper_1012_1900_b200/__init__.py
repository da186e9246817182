"""B200-native gamma-index hot path of arxiv/paper_1012_1900 (Gu, Jia, Jiang).

``binding`` wraps the C-ABI of ``libgamma_b200.so`` (include/gamma_b200.h); ``phantoms`` makes the seeded
synthetic dose grids.  Importing this package does not load the library; the first call does, and fails
loudly if it cannot be built or loaded (there is no CPU fallback).
"""
__all__ = ["binding", "phantoms", "build"]
