"""B200-native per-stage hot path of MHDuet (arXiv 2510.13965) on one uniform ghosted patch.

The product is the C-ABI library built from csrc/ (declared in include/mhd.h); `binding` is the
thin ctypes layer over it and `synth` the seeded input generators. Nothing here imports oracle/.
"""
