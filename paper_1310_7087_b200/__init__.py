"""B200-native checkerboard SU(N) Monte Carlo sweep (hot path of QCDGPU, arxiv 1310.7087).

The product is libqcd_b200.so (hand-written CUDA for sm_100a behind the C ABI of include/qcd.h); this package is
its thin Python binding.  Nothing here computes: there is no CPU fallback.
"""
from .binding import *  # noqa: F401,F403
from .binding import Lattice, QcdError, lib, make_field, qcd_field_t, SYMBOLS, LIB_PATH  # noqa: F401
