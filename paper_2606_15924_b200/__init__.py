"""B200-native sparse-pixel Gaussian-splatting rasteriser (TurboGS hot path, arxiv/paper_2606_15924).

The product is ``libtgs.so`` (hand-written CUDA for sm_100a behind the C ABI of ``include/tgs.h``);
this package is its thin Python binding.  There is no CPU fallback.
"""
from .binding import (Camera, LIB_PATH, PIXELS_ALL, PIXELS_BERNOULLI_ERR, SAMPLE_STATIC_MAX_TILES, SPLAT_WORDS, SYMBOLS,
                      TGS, TgsError, load_library, sample_static)
from .pipeline import SparseIteration, SparseRasterStep

__all__ = ["Camera", "LIB_PATH", "PIXELS_ALL", "PIXELS_BERNOULLI_ERR", "SPLAT_WORDS", "SYMBOLS", "TGS", "TgsError",
           "load_library", "SparseIteration", "SparseRasterStep", "SAMPLE_STATIC_MAX_TILES", "sample_static"]
