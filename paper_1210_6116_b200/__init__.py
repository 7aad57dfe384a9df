"""B200-native Swendsen-Wang sweep of the 2D classical XY model (arXiv 1210.6116).

Thin Python binding over the C-ABI library libxy_b200.so (include/xy.h); every step of the hot
path runs in the CUDA kernels under csrc/.  There is no CPU fallback: importing this package
without the built library, or creating a state without a CUDA device, raises.
"""
from .binding import (XYState, XYError, Obs, PccSchedule, OBS_DTYPE, INIT_COLD, INIT_HOT,
                      FLAG_LABELS64, workspace_bytes, debug_philox, debug_curand_philox, lib_path)

__all__ = ["XYState", "XYError", "Obs", "PccSchedule", "OBS_DTYPE", "INIT_COLD", "INIT_HOT",
           "FLAG_LABELS64", "workspace_bytes", "debug_philox", "debug_curand_philox", "lib_path"]
