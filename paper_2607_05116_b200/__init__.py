"""B200-native routing-trace hot path of CAP (arXiv 2607.05116).

The product is the C-ABI CUDA library declared in include/cap.h; `cap` is its thin
ctypes binding (argument marshalling only).  Importing this package does not load the
library; the first call does, and fails loudly if it is missing.
"""
__all__ = ["cap", "workload"]
