"""paper_1307_7820_b200 -- B200-native two-vector Four-Russians RNA fold (arxiv 1307.7820).

The product is the C-ABI shared library `librna4r.so` (include/rna4r.h) built from csrc/*.cu
for sm_100a; this package is its thin Python binding (argument marshalling only).
"""
from . import shard
from .binding import (ENGINE_AUTO, ENGINE_DIAG, ENGINE_MAXPLUS, ENGINE_PAPER_TILE, ENGINE_SMEM, ENGINE_TILED, TABLE_INT16, TABLE_INT32, TABLE_NONE, Rna4r, Rna4rError,
                      load, rna4r_prepare)

__all__ = ["Rna4r", "Rna4rError", "rna4r_prepare", "load", "TABLE_NONE", "TABLE_INT16", "TABLE_INT32",
           "ENGINE_AUTO", "ENGINE_TILED", "ENGINE_DIAG", "ENGINE_SMEM", "ENGINE_PAPER_TILE", "ENGINE_MAXPLUS", "shard"]
