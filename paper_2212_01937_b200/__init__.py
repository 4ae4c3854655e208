"""B200-native batched LCDM+radiation cosmography (arXiv:2212.01937 hot path).

`paper_2212_01937_b200.binding` is the thin Python layer over the C-ABI library
(include/cosmo_b200.h); `paper_2212_01937_b200.workloads` holds the seeded input generators.
Nothing is imported eagerly so that the generators stay usable without the CUDA library.
"""
__version__ = "0.1.0"
