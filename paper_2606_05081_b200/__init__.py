"""blest-b200: B200-native (sm_100a) BLEST hot path -- BFS / multi-source BFS / closeness over a Binarized
Virtual Slice Set, behind the C ABI of ``include/blest.h``.  See DESIGN.md.

``binding`` is a thin ctypes layer (argument marshalling only); the product is ``libblest.so``.
"""
from .binding import (BlestError, Graph, Info, barrier_microbench, closeness_from_sums, cluster_microbench,  # noqa: F401
                      contraction_selftest, get_vi, l2_microbench, load, mma_microbench, noalloc_limits, strerror, tcgen05_microbench)

__all__ = ["BlestError", "Graph", "Info", "barrier_microbench", "closeness_from_sums", "cluster_microbench", "contraction_selftest",
           "get_vi",
           "l2_microbench", "load", "mma_microbench", "noalloc_limits", "strerror", "tcgen05_microbench"]
