"""B200-native fp64 VL+CT ideal-MHD time step (arxiv 2402.05240, Cholla-MHD hot path).

`paper_2402_05240_b200.mhd` is the thin ctypes binding of the C-ABI CUDA library
(include/mhd.h, csrc/); `paper_2402_05240_b200.inputs` holds the seeded input recipes.
Importing this package does not load the CUDA library; importing `.mhd` does and fails
loudly if it is missing.
"""
__all__ = ["inputs"]
