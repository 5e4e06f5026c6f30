"""B200-native hot path of arXiv 1111.6288: applying the overlap Dirac operator
D_ov = 1 + gamma5 sign(H_w) -- Wilson kernel, Clenshaw polynomial sign, small-space
projector, BLAS-1, multi-shift CG, Lanczos low modes -- as hand-written CUDA for sm_100a behind a C ABI
(include/ov.h).  This package is the thin Python binding (argument marshalling only).
"""
from .binding import (  # noqa: F401
    LIB_PATH,
    SYMBOLS,
    Overlap,
    OvError,
    blas_dot_static,
    blas_dot_static_max,
    chebyshev_coeffs,
    host_eigh,
    load_library,
)
