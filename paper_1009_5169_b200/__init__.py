"""B200-native (sm_100a) blocked Wilson-Dirac solve + fermion force of arxiv/paper_1009_5169.

The product is the C-ABI library `libwd.so` (include/wd.h, sources in csrc/); `wd` is its thin
ctypes binding.  Build with `python -m paper_1009_5169_b200.build`.
"""
from . import wd  # noqa: F401
from .wd import (BC_PERIODIC, BC_SF, F32, F64, LINK12, LINK18, OP_D, OP_DDAG, ORDER_LINEAR,  # noqa: F401
                 ORDER_TILED, OPT_HOP32_SITES, OPT_HOP64_SITES, OPT_HOP32_REGS, OPT_HOP64_REGS, OPT_POLL_EVERY, OPT_HOP_IMPL, OPT_ALTERNATE_SWEEP, OPT_HOP_ROWS, OPT_SOLVER, OPT_PAIRED, OPT_GRAPH, OPT_MERGE, F32P, SOLVER_DC_F32, SOLVER_RELIABLE_H16, SOLVER_GL_FLEX, SOLVER_GL_F64, SOLVER_BL_F64,
                 ACTION_FULL, ACTION_EO, PARITY_EVEN, PARITY_ODD, PARITY_BOTH,
                 Context, WdError, action_static)
