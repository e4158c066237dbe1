"""B200-native (sm_100a) short-range molecular dynamics hot path of arXiv 2003.14061 (Rapaport).

The product is the C-ABI library `libmd_b200.so` (include/md_b200.h, sources in csrc/); this package is its
thin Python binding.  Build with `python -m paper_2003_14061_b200.build`.
"""
from .binding import (Energies, MDError, MDSystem, load_library, use_torch_allocator, velocity_sums_noalloc, NOALLOC_MAX_ATOMS, EXPORTS, LIB_PATH, FLAG_NO_GRAPH, FLAG_GLOBAL_W, FLAG_TILED_W, FLAG_GATHER_W, FLAG_W_TRANSPOSED, FLAG_LAYER_H, FLAG_NO_PERSIST,
                      TIMER_NAMES)

__all__ = ["Energies", "MDError", "MDSystem", "load_library", "use_torch_allocator", "velocity_sums_noalloc", "NOALLOC_MAX_ATOMS", "EXPORTS", "LIB_PATH",
           "TIMER_NAMES"]
