"""B200-native hot path of arXiv:1706.01420 (Ipanema-beta): unbinned fp64 Ipatia + exponential NLL.

Thin Python binding (argument marshalling only) over the C-ABI CUDA library `libipanll.so`
(include/ipanll.h).  Every step of the path runs in the library's sm_100a kernels; there is no
CPU fallback: importing works without a GPU (the library loads, symbols resolve), calling a
compute entry point without one raises.
"""
from .binding import *  # noqa: F401,F403
from .binding import __all__  # noqa: F401
