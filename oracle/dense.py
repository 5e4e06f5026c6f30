"""ORACLE (test infrastructure only): dense brute force on tiny lattices (O9).

The matrix of H_w is built column by column by applying the oracle's own H_w to unit vectors, then
numpy.linalg.eigh gives the exact matrix sign  sign(H_w) = Z sign(Lambda) Z^dagger  -- the plain
definition that the polynomial + small space of PAPER.md:31-39 approximates.
"""
from __future__ import annotations

import numpy as np

from . import capi


def dense_hw(dims, kappa, U) -> np.ndarray:
    X, Y, Z, T = dims
    N = X * Y * Z * T * 12
    H = np.empty((N, N), dtype=np.complex128)
    e = np.zeros(N, dtype=np.complex128)
    for j in range(N):
        e[j] = 1.0
        H[:, j] = capi.hw(dims, kappa, U, e.reshape(T, Z, Y, X, 4, 3)).reshape(N)
        e[j] = 0.0
    return H


def eig_hw(dims, kappa, U):
    """(eigenvalues ascending, eigenvectors as columns) of the Hermitian H_w."""
    H = dense_hw(dims, kappa, U)
    herm_defect = np.max(np.abs(H - H.conj().T))
    w, Zv = np.linalg.eigh(0.5 * (H + H.conj().T))
    return w, Zv, H, herm_defect


def exact_sign_apply(w, Zv, x) -> np.ndarray:
    """sign(H_w) x = Z sign(Lambda) Z^dagger x."""
    shape = x.shape
    v = x.reshape(-1)
    return (Zv @ (np.sign(w) * (Zv.conj().T @ v))).reshape(shape)


def lowest_modes(w, Zv, norm, k, spinor_shape):
    """The k eigenpairs of Q = H_w/norm with smallest |lambda| (reading G12); V as [k] + spinor_shape."""
    idx = np.argsort(np.abs(w))[:k]
    lam = w[idx] / norm
    V = np.ascontiguousarray(Zv[:, idx].T).reshape((k,) + tuple(spinor_shape))
    return V, lam
