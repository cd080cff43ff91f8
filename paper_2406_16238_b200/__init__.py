"""B200-native phaseless-AFQMC walker step (arXiv 2406.16238 hot path).

`paper_2406_16238_b200.afqmc` is the ctypes binding of the C-ABI library
(include/afqmc.h); `paper_2406_16238_b200.inputs` holds the seeded input generators.
Nothing here falls back to a CPU implementation: without the CUDA library the binding
raises at load time.
"""
__all__ = ["inputs", "afqmc"]
