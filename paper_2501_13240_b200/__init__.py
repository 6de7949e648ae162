"""semb200: B200-native (sm_100a, fp64) spectral-element Poisson/Helmholtz hot path.

`inputs` (numpy, seeded synthetic meshes/fields) imports without CUDA.  The operator API lives in
`paper_2501_13240_b200.semb` (ctypes binding over csrc/libsemb200.so) and fails loudly when the
CUDA library is missing; there is no CPU fallback.
"""
__all__ = ["inputs", "semb"]
