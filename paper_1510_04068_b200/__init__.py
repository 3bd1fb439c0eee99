"""B200-native direct N-body force library (hot path of arXiv:1510.04068, Sapporo2).

The product is the C-ABI CUDA library ``libs2b200.so`` (include/s2b200.h); this package is its
thin ctypes binding.  See DESIGN.md.
"""
from .binding import *  # noqa: F401,F403
from .binding import (S2Error, header_symbols, lib, LIB_PATH, s2_ctx)  # noqa: F401
