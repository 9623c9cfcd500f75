"""B200-native exhaustive Ising enumeration (hot path of arXiv 1904.03621).

The product is the C-ABI library declared in include/ising.h, built from csrc/ for sm_100a;
`paper_1904_03621_b200.binding` is the thin ctypes layer over it (argument marshalling only).
Importing this package does not load the CUDA library; the first call does, and fails loudly
if it is missing. There is no CPU fallback.
"""
__all__ = ["binding", "instances"]
