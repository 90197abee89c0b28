"""B200-native checkerboard Cellular Potts sweep (arXiv 2312.09317): thin Python binding over the
C-ABI CUDA library (include/cpm.h).  Argument marshalling only -- every step of the path runs in
the sm_100a kernels under csrc/.  There is no CPU fallback: without the built library or without
a CUDA device the calls fail loudly."""
from .binding import (  # noqa: F401
    CPM, CPMError, MODE_DETERMINISTIC, MODE_LIVE_ATOMICS, FLAG_WARP_KERNEL, FLAG_NO_TMA, FLAG_NO_GRAPH, load_library, library_path, debug_philox,
    exported_symbols, noalloc_setup, NOALLOC_MAX_SITES, NOALLOC_MAX_BINS,
)
