"""chaoticus-b200: B200-native (sm_100a, FP64) hot path of arXiv 2507.00622 ("Chaoticus").

The product is the C-ABI library built from csrc/ (see include/chaoticus.h); `binding`
is a thin ctypes layer with the same entry-point names.  Importing this package does not
load the library; the first call does, and fails loudly if it is missing (there is no CPU
fallback).
"""
__all__ = ["binding", "workloads"]
