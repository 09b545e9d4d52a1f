"""B200-native TPC sector tracking (arxiv/paper_2601_20569).

``paper_2601_20569_b200.binding`` is the thin ctypes layer over the C-ABI library
``libtpctrack.so`` (include/tpc_track.h); ``paper_2601_20569_b200.datagen`` the seeded
input generator.  Importing this package loads nothing; the binding raises if the CUDA
library has not been built (there is no CPU fallback).
"""
__all__ = ["binding", "datagen", "build"]
