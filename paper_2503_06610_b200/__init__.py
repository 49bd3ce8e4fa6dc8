"""B200 (sm_100a) hot path of arXiv 2503.06610: D3Q19 shifted-population lattice Boltzmann +
finite-difference director update, behind the C ABI of include/nh.h.

Only the binding lives here; the kernels are in csrc/ and are compiled by `build.py` into
libnh_b200.so next to this file.  Nothing here imports the CPU oracle.
"""
from .binding import (FP32_SHIFTED, FP32_UNSHIFTED, FP64_SHIFTED, FP64_UNSHIFTED, KERNEL_CLASSES,
                      OPT_CHECK_FINITE, OPT_FD_DIRECT, OPT_FD_NOVEC, OPT_GRAPH, OPT_LB_ONESTEP, OPT_LB_TWOSTEP, OPT_NO_SERPENTINE, OPT_TIMING, TUNE, Lattice, NhError, NhParams,
                      lb_two_steps_noalloc, load, make_params, workspace_bytes)

__all__ = ["Lattice", "NhError", "NhParams", "load", "make_params", "workspace_bytes", "lb_two_steps_noalloc",
           "FP64_SHIFTED", "FP32_SHIFTED", "FP32_UNSHIFTED", "FP64_UNSHIFTED",
           "OPT_GRAPH", "OPT_TIMING", "OPT_FD_DIRECT", "OPT_NO_SERPENTINE", "OPT_FD_NOVEC", "OPT_LB_TWOSTEP", "OPT_LB_ONESTEP", "OPT_CHECK_FINITE", "KERNEL_CLASSES", "TUNE"]
