"""B200-native LLOID multirate SVD matched filtering (arxiv/paper_2511_04730, Sec. II.C-II.D.1).

The product is the C-ABI library ``liblloid.so`` (include/lloid.h, sources in csrc/); this package is its thin
ctypes binding.  Import fails loudly when the library has not been built -- there is no CPU fallback.
"""
from .binding import *  # noqa: F401,F403
from .binding import (EXPORTS, LIB_PATH, PEAK_DTYPE, LloidError, LloidStream, Whitener, bank_slices)  # noqa: F401
