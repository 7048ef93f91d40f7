"""B200-native masked rasterization (MaskGaussian, arXiv 2412.20522) -- hot path only.

`binding` is the thin ctypes layer over the C-ABI library (include/mg.h); `scenes` holds the
seeded synthetic input generators.  Nothing here imports oracle/.
"""
