"""B200-native (sm_100a) hot path of IRIS-SO (arxiv/paper_2607_01338): thin Python binding over the
C-ABI CUDA library declared in include/iris_so.h.  PyTorch is used only for device memory and streams.

The library is loaded lazily on first use; there is no CPU fallback -- a missing or unloadable
libiris_so.so raises, it never degrades to another implementation.
"""
from .binding import (IrisSO, IrisSOError, lib_path, load_library, DECLARED_SYMBOLS,
                      ALGO_AUTO, ALGO_DENSE, ALGO_WINDOW, ALGO_WINDOW_EDGE)

__all__ = ["IrisSO", "IrisSOError", "lib_path", "load_library", "DECLARED_SYMBOLS",
           "ALGO_AUTO", "ALGO_DENSE", "ALGO_WINDOW", "ALGO_WINDOW_EDGE"]
