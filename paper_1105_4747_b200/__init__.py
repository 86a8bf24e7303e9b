"""B200-native Lya-forest tau/F/A hot path of arXiv:1105.4747.

`lya` (the ctypes binding over the C-ABI library include/lya.h) is imported lazily so
that the input generator and workload tables stay usable without the CUDA library.
"""
from .workloads import WORKLOADS, Workload, scaled  # noqa: F401
