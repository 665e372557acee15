"""paper_2503_09629_b200 — B200-native (sm_100a) subcycled RK4 AMR step with dense-output ghost fill.

The product is ``libsubcycle.so`` (C ABI in ``include/subcycle.h``, CUDA sources in ``csrc/``); this
package is its thin Python binding plus the seeded synthetic workloads. Nothing here imports ``oracle/``.
"""
from . import workloads  # noqa: F401
from .binding import (EXPORTS, Hierarchy, SubcycleError, lib, make_desc, sc_arena_bytes,  # noqa: F401
                      sc_box, sc_hierarchy_desc, sc_max_abs_noalloc, SC_NOALLOC_MAX_DOUBLES,
                      sc_debug_interp_weights)
