"""B200-native Swendsen-Wang sweep of the 2D classical XY model (arXiv 1210.6116).

Thin Python binding over the C-ABI library libxy_b200.so (include/xy.h); every step of the hot
path runs in the CUDA kernels under csrc/.  There is no CPU fallback: touching any name of the
binding without the built library, or creating a state without a CUDA device, raises.

The binding is loaded on first use so that `paper_1210_6116_b200.build` (which produces the
library) can be imported before the library exists.
"""
__all__ = ["XYState", "XYError", "Obs", "PccSchedule", "OBS_DTYPE", "INIT_COLD", "INIT_HOT", "OBS_NONE", "OBS_ALL",
           "FLAG_LABELS64", "FLAG_FOURIER", "Fourier", "FOURIER_DTYPE", "workspace_bytes", "debug_philox", "debug_check_counts", "debug_curand_philox", "lib_path",
           "PottsState", "PottsObs", "SlabState", "PccState", "observe_static", "xi2nd"]


def __getattr__(name):
    if name in __all__:
        from . import binding
        return getattr(binding, name)
    raise AttributeError(f"module {__name__!r} has no attribute {name!r}")
