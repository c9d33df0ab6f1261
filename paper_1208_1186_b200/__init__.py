"""paper_1208_1186_b200 -- B200-native Landau gauge fixing (steepest descent + Fourier acceleration)
of 4D SU(3) lattice gauge fields, arXiv 1208.1186.

The product is the C-ABI library `liblgf.so` (include/lgf.h, csrc/*.cu, hand-written CUDA for
sm_100a).  This package is a thin ctypes binding with the same names; torch is used only for
device memory and streams.  There is no CPU fallback: without the built library or without a CUDA
device every call raises.
"""
from .binding import (  # noqa: F401
    LGF_F32, LGF_F64, LGF_REAL12, LGF_REAL18, LGF_HOST, LGF_DEVICE,
    GaugeFixer, LgfError, LgfResult, library_path, load_library, declared_symbols, workspace_bytes,
    measure_static, static_init, STATIC_MAX_SITES,
)
