"""B200-native chi0*dV hot path of arXiv 2203.05623 (batched Gamma-point Sternheimer): Python face of libwest.so.

The product is the C-ABI library declared in include/west.h (hand-written sm_100a kernels); this package only loads it
and marshals arguments.  Build it in-tree with ``python -m paper_2203_05623_b200.build``.
"""
from .binding import (  # noqa: F401
    EXPORTS, LIB_PATH, WEST_FP32, WEST_FP64, WEST_FP64_I8, WEST_FULL, WEST_GAMMA, WEST_MIXED, WEST_NOTCONVERGED, WEST_OK, West, WestError, load_library,
    west_cell, west_cg_opts, west_stats,
)
