"""paper_1409_4256_b200: one EMC iteration (arXiv 1409.4256) on one B200, as hand-written sm_100a
CUDA behind a C ABI (include/emc.h, csrc/) with a thin ctypes binding of the same names."""
from . import binding
from .binding import *  # noqa: F401,F403  (binding.__all__: the emc_* calls, EMC_* constants and helpers)

__all__ = list(binding.__all__)
