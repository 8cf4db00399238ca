"""B200-native ALE Galerkin-Boltzmann nodal-DG + SARK4 stage library (arxiv/paper_2607_00199 hot path).

The product is the C-ABI shared library ``libalegb.so`` (include/alegb.h; sources in csrc/); ``binding`` is a thin
ctypes layer over it.  There is no CPU or PyTorch fallback: importing ``binding`` without the built library raises.
"""
