"""paper_1409_8336_b200 — B200-native condensed-history proton Monte Carlo (hot path of arxiv 1409.8336).

The product is libpmc.so (CUDA, sm_100a) behind the C-ABI of include/pmc.h; this package is its thin binding.
"""
from .binding import Pmc, PmcError, load_library, LIB_PATH, EXPORTS, SECONDARY_DTYPE  # noqa: F401
from .build import build  # noqa: F401
