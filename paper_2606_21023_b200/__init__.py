"""B200-native HEAL compensated GEMM (arxiv/paper_2606_21023, Eq. 10).

The product is the C-ABI library ``libheal.so`` (include/heal.h, csrc/); ``binding`` is the thin
ctypes layer over it (argument marshalling only).  Importing this package does not load the
library; the first call does, and fails loudly if it is missing.
"""
__all__ = ["binding", "inputs"]
