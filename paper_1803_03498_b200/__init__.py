"""B200-native HEOM right-hand side + RK4 (arXiv 1803.03498, DM-HEOM hot path).

`Heom` mirrors the C ABI in include/heom.h.  The CUDA library is loaded on first
use and its absence is an error: there is no CPU fallback in this package.
"""
from .binding import Heom, HeomError, load_library, LIB_PATH, SYMBOLS, level_max_static, STATIC_MAX_DEPTH  # noqa: F401
