"""B200-native hot path of transport DPD with explicit RBC membranes (arXiv:1611.06163): libtdpd.so (hand-written
CUDA for sm_100a behind the C ABI of include/tdpd.h) and its thin ctypes binding.  No CPU fallback."""
from .binding import (LIB_PATH, SYMBOLS, TIMER_NAMES, Params, RbcParams, Simulation, TdpdError, load_library, host_grid,
                      make_params, make_rbc_params, measure_peaks, noalloc_init, sort_cells_noalloc, NOALLOC_MAX_N)

__all__ = ["LIB_PATH", "SYMBOLS", "TIMER_NAMES", "Params", "RbcParams", "Simulation", "TdpdError", "load_library", "host_grid",
           "make_params", "make_rbc_params", "measure_peaks", "noalloc_init", "sort_cells_noalloc", "NOALLOC_MAX_N"]
