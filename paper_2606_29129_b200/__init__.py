"""paper_2606_29129_b200 -- B200-native DGEMM emulation by Ozaki scheme II on INT8 tensor cores.

The product is the C-ABI library libozaki2.so (include/ozaki2.h, sources under csrc/); this package is its
thin Python binding.  Import is light: the library is loaded on first use and there is no fallback.
"""
from .binding import *  # noqa: F401,F403
from .binding import lib, Ozaki2Error  # noqa: F401
