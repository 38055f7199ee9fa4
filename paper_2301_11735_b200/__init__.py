"""B200-native coupled-pair Metropolis sweep of arXiv:2301.11735 (charge-conserving parallel Monte Carlo).

The product is the C-ABI library `libic_b200.so` (include/ic.h; sources in csrc/, hand-written sm_100a CUDA).
`binding` exposes the same entry points through ctypes; `Sim` is a convenience wrapper that uses PyTorch only for
device memory and the stream; `scan.temperature_scan` is the C(T), chi(T) driver on top of it.
"""
from .binding import (IC_ERR_CHARGE, IC_ERR_CUDA, IC_ERR_NULL, IC_ERR_PARAM, IC_ERR_SIZE, IC_ERR_WORKSPACE,  # noqa: F401
                      IC_ERR_STATIC_MAX, IC_N_CLASSES, IC_OK, IC_STATIC_CLUSTER_MAX_L, EXPORTS, LIB_PATH, IcError, Sim, ic_obs,
                      largest_cluster_static, lib)
