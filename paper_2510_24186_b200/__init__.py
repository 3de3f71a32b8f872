"""tridsk: B200-native (sm_100a) batched gradient-guided Monte Carlo docking kernel library.

The product is the C-ABI shared library ``libtridsk.so`` (include/tridsk.h, csrc/); this package
is its thin ctypes binding.  Build it in-tree with ``python -m paper_2510_24186_b200.build``.
"""
from .binding import (Engine, Grid, Ligands, Params, TridskError, TRACE_DTYPE, default_params, lib, split_state,
                      LIB_PATH)

__all__ = ["Engine", "Grid", "Ligands", "Params", "TridskError", "TRACE_DTYPE", "default_params", "lib",
           "split_state", "LIB_PATH"]
