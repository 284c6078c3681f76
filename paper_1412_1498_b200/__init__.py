"""paper_1412_1498_b200 — B200-native (sm_100a) overrelaxation gauge fixing, the hot path of arXiv:1412.1498.

The product is the C-ABI library libgf.so (include/gf.h, csrc/); this package is its thin Python binding.
"""
from .binding import *  # noqa: F401,F403
from .binding import GaugeFixer, GFError, SYMBOLS  # noqa: F401
from .sharded import GpuSlabEngine, ShardedGaugeFixer  # noqa: F401
