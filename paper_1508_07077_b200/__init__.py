"""B200-native (sm_100a) implicit-depletant hard-particle Monte Carlo: the checkerboard colloid trial move of
arXiv 1508.07077.  Thin Python binding over the C-ABI library declared in include/hpmc.h; every step of the path
runs in the library's CUDA kernels.  There is no CPU fallback: loading fails loudly if the library is missing.
"""
from .binding import HPMC, Params, COUNTER_NAMES, SHAPES, OPT_SHELL, OPT_ROSENBLUTH, load_library, HPMCError, alu_peaks, cells_noalloc  # noqa: F401
