"""B200-native bump x load effective-resistance analysis of 3D-IC PDNs (arxiv/paper_2607_05818).

The product is the CUDA library `libpdn.so` (sources in csrc/, C ABI in include/pdn.h); this
package is its thin Python binding.  Importing the package does not load the library; the first
use does, and fails loudly if it has not been built (`__graft_entry__.build()`).
"""
from .binding import (KERNEL_CLASSES, LIB_PATH, PDN_NO_UNIFORM_FAST_PATH, PDN_SKIP_CONNECTIVITY_CHECK,  # noqa: F401
                      PDN_NO_INITIAL_GUESS, PDN_PRECOND_F32, PDN_STATIC_MAX_LOADS, PDN_TERMINAL_PAIRS,
                      PDN_TIERS_ON_HOST,
                      PDN_TIME_KERNELS, EXPORTS, Pdn, PdnError, load_library, shard_bounds)
