"""SCAPE (arXiv 2607.01678) per-shard sparse optimizer step, B200-native.

The product is `libscape.so` (C-ABI in include/scape.h, CUDA kernels for sm_100a under csrc/).
`binding` is the thin ctypes layer with the same names; `synth` holds the seeded synthetic
input generators (no method arithmetic).  Nothing here imports oracle/.
"""
__all__ = ["binding", "synth", "build"]
