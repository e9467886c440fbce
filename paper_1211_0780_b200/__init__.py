"""B200-native Monte Carlo step of the 3-D XY model over parallel-tempering replicas
(arXiv:1211.0780): checkerboard Metropolis + over-relaxation sweeps, observable reduction,
replica exchange -- hand-written sm_100a CUDA behind a C ABI (include/xy.h).

`inputs` (seeded synthetic workloads) imports without the CUDA library; everything else
loads paper_1211_0780_b200/libxy_b200.so on first use and fails loudly if it is missing.
"""
from . import inputs  # noqa: F401

__all__ = ["inputs", "XY", "load_library", "build_library"]


def __getattr__(name):
    if name in ("XY", "load_library", "XYError", "measure_static", "debug_sincos", "debug_sincos64", "debug_atan2", "debug_philox"):
        from . import binding
        return getattr(binding, name)
    if name == "build_library":
        from .build import build_library
        return build_library
    raise AttributeError(name)
