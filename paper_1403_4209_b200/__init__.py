"""B200-native convolutional gridding with W-projection (arXiv 1403.4209 hot path).

`synth` holds the seeded input generators; `binding` is the thin ctypes layer
over the C-ABI library `libig.so` (include/ig.h). Nothing is loaded at import
time; `binding.load()` fails loudly if the CUDA library has not been built.
"""
__all__ = ["synth", "binding", "build"]
