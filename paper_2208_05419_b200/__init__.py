"""B200-native AFNO spectral token-mixing layer (FourCastNet, arXiv 2208.05419).

The product is the C-ABI library built from csrc/ (include/afno.h) and the thin binding in
`binding.py`.  Importing the package does not load the CUDA library; the first call does and
fails loudly if it is missing (there is no CPU fallback).
"""
__all__ = ["binding", "inputs", "build"]
