"""B200-native TPC sector CA tracker: thin Python binding of the tpcca C-ABI library.

The package holds the CUDA sources (csrc/), the in-tree build (build.py) and the ctypes binding
(binding.py).  All five stages of the hot path run in the kernels of libtpcca.so; Python only
marshals arguments.  PyTorch lends device memory (the workspace) and the stream.  There is no
CPU fallback: without the built library or without a CUDA device every entry point raises.
"""
from .binding import (TpccaError, Tracker, Pipeline, SectorOutput, load_library, library_path, abi_symbols, start_hits_noalloc,
                      STAGE_GRID, STAGE_NEIGHBOURS, STAGE_CLEAN, STAGE_START, STAGE_TRACKLETS, STAGE_ALL, STAGE_SELECT, STAGE_RESIDUALS, STAGE_MERGE)

__all__ = ["TpccaError", "Tracker", "Pipeline", "SectorOutput", "load_library", "library_path", "abi_symbols", "start_hits_noalloc",
           "STAGE_GRID", "STAGE_NEIGHBOURS", "STAGE_CLEAN", "STAGE_START", "STAGE_TRACKLETS", "STAGE_ALL", "STAGE_SELECT", "STAGE_RESIDUALS", "STAGE_MERGE"]
