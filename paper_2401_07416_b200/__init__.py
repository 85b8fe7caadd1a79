"""paper_2401_07416_b200 -- B200-native FDTD/TDSE hot path of arXiv 2401.07416.

The product is libtdse.so (csrc/, C ABI in include/tdse.h); this package is the thin Python
binding over it.  There is no CPU fallback.
"""
from .binding import (Tdse, TdseError, load, LIB_PATH, SYMBOLS, dissimilarity_static, TDSE_STATIC_SCRATCH_DOUBLES,
                      TDSE_F32, TDSE_F64, TDSE_BC_PERIODIC, TDSE_BC_DIRICHLET,
                      TDSE_OK, TDSE_EINVAL, TDSE_ENOMEM, TDSE_ECUDA, TDSE_ESTATE, TDSE_EUNSTABLE,
                      TDSE_KERNEL_AUTO, TDSE_KERNEL_TWOPASS, TDSE_KERNEL_FUSED)
from .build import build

__all__ = ["Tdse", "TdseError", "load", "build", "LIB_PATH", "SYMBOLS", "dissimilarity_static"]
