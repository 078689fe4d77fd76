"""sqeq-b200: B200-native periodic Coulomb (cell-list neighbour build, erfc real-space
sum, smooth PME) for the shadow charge-equilibration MD of arxiv 2503.21176.

The product is the C-ABI library built from csrc/ (see include/sqeq.h); `binding`
is the thin ctypes layer with the same names.  Importing this package does not
load the CUDA library; `binding.load()` does, and fails loudly if it is missing.
"""
__all__ = ["binding", "workloads"]
