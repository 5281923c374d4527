"""B200-native thermochemistry hot path of arXiv 2503.24286 (Pyrometheus).

`paper_2503_24286_b200.binding` is the thin ctypes layer over the C-ABI library
`libpyro.so` (include/pyro.h); `paper_2503_24286_b200.inputs` draws the seeded
synthetic mechanisms and states.  Importing the package does not load CUDA.
"""
__all__ = ["binding", "inputs"]
