"""pinmpc — B200-native batched ADMM-MPC solver (hot path of arxiv/paper_2606_05687, pi^n MPC).

`binding` is a thin ctypes layer over libpinmpc.so (include/pinmpc.h); all arithmetic runs in
hand-written CUDA kernels for sm_100a (csrc/).  No CPU fallback.
"""
from . import binding  # noqa: F401
from .binding import (METHOD_AUTO, METHOD_DENSE, METHOD_SRB, NX, LandmarkCfg, Landmarks, Layout,  # noqa: F401
                      PinmpcError, Solver, SplitSolver, make_landmark_cfg, make_layout)
