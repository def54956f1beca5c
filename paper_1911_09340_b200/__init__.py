"""B200-native seed x hit scan of arXiv 1911.09340 (COMET Phase-I multi-turn reconstruction).

The product is the C-ABI library `libcomet.so` (include/comet.h); `binding` marshals torch tensors
into it.  Nothing here has a CPU implementation: without the built library, or without a CUDA
device, the calls raise.
"""
from .binding import Comet, CometError, argmin_static, lib_path, load_library, EXPORTED_SYMBOLS

__all__ = ["Comet", "CometError", "argmin_static", "lib_path", "load_library", "EXPORTED_SYMBOLS"]
