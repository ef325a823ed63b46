"""B200-native fp64 geometric multigrid for the variable-density pressure Poisson
equation of a two-phase VOF projection step (arxiv/paper_2605_30082's FS3D hot path).

Everything numerical runs in the hand-written sm_100a kernels of ``csrc/`` behind the C
ABI of ``include/mg.h``; this package is the thin ctypes binding with the same names.
There is no CPU fallback: importing :mod:`.binding` without a loadable libmg raises.
"""
from .binding import (  # noqa: F401
    MG_BC_NEUMANN,
    MG_BC_PERIODIC,
    MgError,
    Multigrid,
    lib,
    residual_norm_static,
    workspace_bytes,
)
