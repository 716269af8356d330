"""B200-native checkerboard heat-bath / overrelaxation / parallel-tempering sweeps of the 3d
anisotropic Heisenberg spin glass (arXiv:1309.1599).  The product is the C-ABI library
libsg_b200.so (include/sg_b200.h); this package is its thin ctypes binding."""
from .binding import (SpinGlass, SgError, load_library, chiral_cross_static, SG_ELIMIT, STATIC_SCRATCH_BYTES, correlation_length, walk_tau_int, GEN_OFFDIAG_SYM, GEN_PAPER_SYM6, GEN_GENERAL9,
                      GEN_BIMODAL, GEN_FERRO, KIND_OR, KIND_HB, DECLARED_SYMBOLS, TUNE_SWEEP_IMPL, TUNE_ZCHUNK, TUNE_RES_COPIES, TUNE_PACKED, TUNE_MEASURE_IMPL, TUNE_GRAPH, TUNE_CLUSTER_CTAS, MEASURE_AUTO, MEASURE_STAGED, LOGBINS,
                      SWEEP_AUTO, SWEEP_TILED, SWEEP_ZMARCH, SWEEP_RESIDENT, SWEEP_FUSED, SWEEP_CLUSTER)

__all__ = ["SpinGlass", "SgError", "load_library", "chiral_cross_static", "SG_ELIMIT", "STATIC_SCRATCH_BYTES", "correlation_length", "walk_tau_int", "GEN_OFFDIAG_SYM", "GEN_PAPER_SYM6", "GEN_GENERAL9",
           "GEN_BIMODAL", "GEN_FERRO", "KIND_OR", "KIND_HB", "DECLARED_SYMBOLS", "TUNE_SWEEP_IMPL", "TUNE_ZCHUNK", "TUNE_RES_COPIES", "TUNE_PACKED", "TUNE_MEASURE_IMPL", "TUNE_GRAPH", "TUNE_CLUSTER_CTAS", "MEASURE_AUTO", "MEASURE_STAGED", "LOGBINS",
           "SWEEP_AUTO", "SWEEP_TILED", "SWEEP_ZMARCH", "SWEEP_RESIDENT", "SWEEP_FUSED", "SWEEP_CLUSTER"]
