"""B200-native Wannier-to-Bloch interpolation of electron-phonon matrix elements (arxiv/paper_2603_10295).

The product is the CUDA library `libepw_interp.so` (sources in csrc/, C ABI in include/epw_interp.h);
this package is its thin Python binding.  Nothing here imports `oracle/`.
"""
from .binding import *  # noqa: F401,F403
from .binding import EpwError, EpwInterp, load_library  # noqa: F401
