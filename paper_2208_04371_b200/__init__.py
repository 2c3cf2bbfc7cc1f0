"""B200-native explicit Yee FDTD hot path of the ARTEMIS S-parameter workflow (arXiv 2208.04371).

The product is the CUDA library libfdtd_b200.so (csrc/, C ABI in include/fdtd.h).  This package is the thin binding:
`binding` mirrors the C ABI name for name, `Solver` wraps a handle and its torch workspace, `sparams` forms S* (Eq. 1-2)
from the port DFTs, renormalises it to 50 ohm (Eq. 5-6) and gives the phase delay (Eq. 8), `nport` runs the paper's
inc/tot protocol over every driving port.  There is no CPU fallback.
"""
from .binding import (FDTD_EX, FDTD_EY, FDTD_EZ, FDTD_F32, FDTD_F64, FDTD_HX, FDTD_HY, FDTD_HZ, FDTD_MAT_FULL,  # noqa: F401
                      FDTD_MAT_INDEXED, FDTD_OPT_FUSED_KZ, FDTD_OPT_FUSED_TILE, FDTD_OPT_GRAPH_UNROLL, FDTD_OPT_STEP_IMPL, FDTD_OPT_TUNE_MEMO, FDTD_OPT_USE_GRAPH, FDTD_OPT_Z_SPIN, FDTD_W_DGAUSS,
                      FDTD_W_GAUSS, FDTD_W_GSINE, FdtdError)
from .solver import Solver  # noqa: F401
