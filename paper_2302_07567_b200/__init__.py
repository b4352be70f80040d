"""B200-native hot path of arXiv 2302.07567 (relativistic space-charge BLDTT-FMM).

The product is the C-ABI library ``libfmm_b200.so`` (``include/fmm.h``); ``binding`` is the
thin Python layer over it.  Importing this package does not load the library: the first call
into ``binding`` does, and fails loudly if the CUDA extension is missing.
"""
__all__ = ["binding", "workloads"]
