"""ORACLE (test infrastructure only): ctypes access to overlap_oracle.c.

All arrays are canonical (workloads/ conventions): gauge [T][Z][Y][X][4][3][3], spinor [T][Z][Y][X][4][3],
complex128, C-contiguous.  dims = (X, Y, Z, T).
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "overlap_oracle.c")
_LIB = os.path.join(_HERE, "liboverlap_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile the C oracle with gcc (building the checker is not using it)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-fopenmp", "-fcx-limited-range", "-std=c99", "-shared", "-fPIC",
               "-o", _LIB, _SRC, "-lm"]
        subprocess.check_call(cmd)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        build()
        _lib = ctypes.CDLL(_LIB)
    return _lib


def num_threads() -> int:
    """OpenMP threads the oracle will use (OMP_NUM_THREADS or all cores)."""
    v = os.environ.get("OMP_NUM_THREADS")
    return int(v) if v else (os.cpu_count() or 1)


def _c(a):
    a = np.ascontiguousarray(a, dtype=np.complex128)
    return a, a.ctypes.data_as(ctypes.c_void_p)


def _d(a):
    a = np.ascontiguousarray(a, dtype=np.float64)
    return a, a.ctypes.data_as(ctypes.c_void_p)


def _dims(dims):
    return (ctypes.c_int * 4)(*[int(d) for d in dims])


BC_DEFAULT = (1.0, 1.0, 1.0, -1.0)   # periodic in space, antiperiodic in time (north_star; G11)


def set_boundary(bc=BC_DEFAULT) -> None:
    """Boundary factor per direction (x, y, z, t) of a hop across the lattice boundary: +1 periodic, -1 antiperiodic,
    0 Dirichlet/open.  Global state of the C oracle; every operator below uses it."""
    arr = (ctypes.c_double * 4)(*[float(v) for v in bc])
    _load().orc_set_boundary(arr)


class boundary:
    """with oracle.boundary((1, 1, 0, 0)): ...   -- sets the boundary factors, restores the default on exit."""

    def __init__(self, bc):
        self.bc = bc

    def __enter__(self):
        set_boundary(self.bc)
        return self

    def __exit__(self, *exc):
        set_boundary(BC_DEFAULT)
        return False


def gamma(idx: int) -> np.ndarray:
    """gamma_x, gamma_y, gamma_z, gamma_t (idx 0..3) or gamma5 (idx 4) as the oracle uses them."""
    out = np.zeros((4, 4), dtype=np.complex128)
    _load().orc_gamma(ctypes.c_int(idx), out.ctypes.data_as(ctypes.c_void_p))
    return out


def wilson_hop(dims, U, psi) -> np.ndarray:
    U, pU = _c(U)
    psi, pp = _c(psi)
    out = np.empty_like(psi)
    _load().orc_wilson_hop(_dims(dims), pU, pp, out.ctypes.data_as(ctypes.c_void_p))
    return out


def hw(dims, kappa, U, psi) -> np.ndarray:
    U, pU = _c(U)
    psi, pp = _c(psi)
    out = np.empty_like(psi)
    _load().orc_hw(_dims(dims), ctypes.c_double(kappa), pU, pp, out.ctypes.data_as(ctypes.c_void_p))
    return out


def sign_poly(dims, kappa, U, coef, eps, norm, x) -> np.ndarray:
    U, pU = _c(U)
    x, px = _c(x)
    coef, pc = _d(coef)
    out = np.empty_like(x)
    _load().orc_sign_poly(_dims(dims), ctypes.c_double(kappa), pU, pc, ctypes.c_int(len(coef) - 1),
                          ctypes.c_double(eps), ctypes.c_double(norm), px,
                          out.ctypes.data_as(ctypes.c_void_p))
    return out


def _small(V, lam):
    if V is None or lam is None or len(lam) == 0:
        return None, None, None, None, 0
    V, pV = _c(V)
    lam, pl = _d(lam)
    return V, pV, lam, pl, len(lam)


def sign(dims, kappa, U, coef, eps, norm, V, lam, x) -> np.ndarray:
    U, pU = _c(U)
    x, px = _c(x)
    coef, pc = _d(coef)
    V, pV, lam, pl, k = _small(V, lam)
    out = np.empty_like(x)
    _load().orc_sign(_dims(dims), ctypes.c_double(kappa), pU, pc, ctypes.c_int(len(coef) - 1),
                     ctypes.c_double(eps), ctypes.c_double(norm), pV, pl, ctypes.c_int(k), px,
                     out.ctypes.data_as(ctypes.c_void_p))
    return out


def dov(dims, kappa, U, coef, eps, norm, V, lam, mass, x) -> np.ndarray:
    U, pU = _c(U)
    x, px = _c(x)
    coef, pc = _d(coef)
    V, pV, lam, pl, k = _small(V, lam)
    out = np.empty_like(x)
    _load().orc_dov(_dims(dims), ctypes.c_double(kappa), pU, pc, ctypes.c_int(len(coef) - 1),
                    ctypes.c_double(eps), ctypes.c_double(norm), pV, pl, ctypes.c_int(k),
                    ctypes.c_double(mass), px, out.ctypes.data_as(ctypes.c_void_p))
    return out
