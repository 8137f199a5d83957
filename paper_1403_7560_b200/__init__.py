"""paper_1403_7560_b200 -- Swendsen-Wang multi-cluster update (arXiv 1403.7560) on one B200.

The product is libsw_b200.so (csrc/, C ABI in include/sw.h); this package builds it in-tree and
exposes the thin ctypes binding.  No CPU fallback exists: without the built CUDA library or a
CUDA device the calls raise."""
from .binding import (CLOCK, ISING, MICRO_GATHER, MICRO_PHILOX_GROUP, MICRO_PHILOX_SITE, POTTS, STATIC_MAX_SITES, XY,  # noqa: F401
                      SwendsenWang, SwError, cluster_stats_static, lib, micro_bench, philox_selftest)
