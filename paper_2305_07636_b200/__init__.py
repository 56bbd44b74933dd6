"""B200-native event-based multigroup time-dependent Monte Carlo transport (hot path of
arxiv 2305.07636).  Thin binding over the C-ABI in include/mcdc.h; every step of the
path runs in the CUDA kernels under csrc/.  There is no CPU fallback."""
from .binding import Problem, McdcError, load_library, batch_stats_noalloc, COUNTER_NAMES, NOALLOC_MAX_BINS  # noqa: F401
