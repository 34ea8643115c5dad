"""B200-native Riccati-parametrised Eilenberger sweep (arXiv 2205.15000 hot path).

Thin Python binding over the C-ABI library `libsc_riccati.so` (include/sc_riccati.h).  Argument
marshalling only: every step of the path runs in the library's CUDA kernels.  PyTorch is used for
device memory and streams.  There is no CPU fallback: importing works anywhere, but creating a context
without the built library or without a CUDA device raises.
"""
from .binding import (ScError, ScContext, SweepStats, lib_path, load_library, declared_symbols,  # noqa: F401
                      sc_residual_norm_static, RESIDUAL_STATIC_MAX_ELEMENTS, SYM_S, SYM_DX2Y2, SYM_DXY, SYM_G)

__all__ = ["ScError", "ScContext", "SweepStats", "lib_path", "load_library", "declared_symbols",
           "sc_residual_norm_static", "RESIDUAL_STATIC_MAX_ELEMENTS",
           "SYM_S", "SYM_DX2Y2", "SYM_DXY", "SYM_G"]
from .ozaki import ozaki_poles, ozaki_energy_table  # noqa: F401,E402
