"""B200-native RT-TDA sigma-vector / propagation library (arXiv 2601.16949 hot path).

The product is the CUDA library librttda.so (csrc/, C-ABI in include/rttda.h); this package is the
thin binding.  It never imports oracle/ and has no CPU fallback.
"""
from .binding import (Rttda, RttdaError, rttda_overlap, rttda_dipole_ao, rttda_fp64_peak, lib, LIB_PATH,
                      EXPORTS, INFO, OPT_INCORE, OPT_GRAPH, OPT_CX_LR, OPT_RS_OMEGA, make_field)

__all__ = ["Rttda", "RttdaError", "rttda_overlap", "rttda_dipole_ao", "rttda_fp64_peak", "lib", "LIB_PATH",
           "EXPORTS", "INFO", "OPT_INCORE", "OPT_GRAPH", "OPT_CX_LR", "OPT_RS_OMEGA", "make_field"]
