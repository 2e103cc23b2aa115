"""B200-native sparse-grid Gross-Pitaevskii hot path (arxiv/paper_2603_05447): Python binding of the
C-ABI library libgpe_b200.so.  See include/gpe.h for the boundary and DESIGN.md for the design."""
from .binding import (C64, C128, DRESSED, HARMONIC, MASK_AT_DELTA0, MASK_AT_DELTA1, MASK_UNION, SYMBOLS,
                      NORM_NOALLOC_MAX_VALUES, OPT_FUSED_K1, OPT_PDL, OPT_RK4_GRAPH,
                      GpeError, Grid, Sim, lib, norm_noalloc)

__all__ = ["C64", "C128", "DRESSED", "HARMONIC", "MASK_AT_DELTA0", "MASK_AT_DELTA1", "MASK_UNION", "SYMBOLS",
           "NORM_NOALLOC_MAX_VALUES", "OPT_FUSED_K1", "OPT_PDL", "OPT_RK4_GRAPH", "GpeError", "Grid", "Sim", "lib", "norm_noalloc"]
