"""uts — B200-native HEALPix spherical Gaussian-splat rasteriser (hot path of arxiv/paper_2606_29794).

`scenes` is importable without the CUDA library; everything in `binding` fails loudly if `libuts.so` is missing.
"""
__all__ = ["scenes", "binding"]
