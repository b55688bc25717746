"""B200-native spectral-element Poisson/Helmholtz hot path (arXiv 2110.01716): w = Q Q^T (D^T G D) u, Jacobi-PCG.

`paper_2110_01716_b200.inputs`  — seeded synthetic meshes / fields (no method arithmetic, no CUDA).
`paper_2110_01716_b200.binding` — thin ctypes binding over the C-ABI library libsem.so (include/sem.h).
"""
__all__ = ["inputs", "binding"]
