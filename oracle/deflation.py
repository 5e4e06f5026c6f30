"""ORACLE (test infrastructure only): low modes of the overlap operator and the deflated multi-mass CG.

PAPER.md:45  "we use deflation to help speed up the calculation.  This consists of computing the low lying spectrum of
              the overlap operator. ... The process of obtaining the eigenmodes for D_ov is similar to the computation
              of the eigenmodes of H_w"
PAPER.md:81  "we can obtain the eigensystems for D_ov which will be used for deflation to help speed up the propagator
              calculations ... Chebyshev order of 12 ... 100 lowest eigenmodes"

The paper gives no formula, so the plain definitions are written out (reading G20):

  * "eigenmodes of D_ov" = eigenpairs (mu, w) of the Hermitian normal operator  A = D_ov(0)^+ D_ov(0) = gamma5 D gamma5 D
    (the operator the multi-mass CG inverts, reading G10).  With S = sign(H_w), S^2 = 1:
        A = (gamma5 + S)^2 = 2 + gamma5 S + S gamma5,    [A, gamma5] = 0,
    so A is block diagonal in chirality.  On a vector of chirality s (gamma5 x = s x, s = +-1)
        A x = 2 x + (s + gamma5) S x                                                    (one sign per application)
    Non-zero eigenvalues (0 < mu < 4) occur once in EACH sector (w_-s ~ (1 - s gamma5) D w_s), zero modes and their
    mu = 4 partners in one sector only; the low modes of A are therefore computed sector by sector (a Krylov method on
    the whole of A would face an exactly doubly degenerate spectrum).
  * deflated solve of (A + sigma_i) x_i = b for all shifts: with W = [w_1 .. w_K] orthonormal eigenvectors of A,
        x_i = sum_j w_j (w_j^+ b) / (mu_j + sigma_i)  +  multishift_cg(A, sigma, b - W W^+ b)_i
    (the Krylov space of the projected source stays orthogonal to W because W is invariant under A).  W must be
    eigenvectors of the SAME A the CG applies, to the CG tolerance: with a polynomial sign of error delta the sector
    form above and gamma5 D gamma5 D differ by 1 - S^2 = O(delta), so deflation is meant for delta <~ tol.

  * chirally symmetric normal operator (reading G22): A' = 2 + gamma5 S + S gamma5 (normal_op_sym).  Same cost as
    gamma5 D gamma5 D for a general vector (two signs), ONE sign (sector_op) for a vector of definite chirality -- e.g. a
    point source in the chiral basis -- and the sector eigenvectors deflate it exactly.

Spinors are canonical arrays [T][Z][Y][X][4][3]; gamma5 = diag(1,1,-1,-1) acts on the spin index (G2).
"""
from __future__ import annotations

import numpy as np

from .multishift_cg import multishift_cg


def gamma5(x: np.ndarray) -> np.ndarray:
    out = np.array(x, dtype=np.complex128, copy=True)
    out[..., 2:, :] *= -1.0
    return out


def chiral_project(x: np.ndarray, s: int) -> np.ndarray:
    """P_s x = (1 + s gamma5)/2 x."""
    return 0.5 * (x + s * gamma5(x))


def normal_op(apply_dov0, x: np.ndarray) -> np.ndarray:
    """A x = gamma5 D_ov(0) gamma5 D_ov(0) x  -- the plain definition (two applications of D_ov)."""
    return gamma5(apply_dov0(gamma5(apply_dov0(x))))


def sector_op(apply_sign, s: int, x: np.ndarray) -> np.ndarray:
    """A_s x = 2 x + (s + gamma5) sign(H_w) x  for x of chirality s (one application of the sign)."""
    y = apply_sign(x)
    return 2.0 * x + s * y + gamma5(y)


def normal_op_sym(apply_sign, x: np.ndarray) -> np.ndarray:
    """A' x = 2 x + gamma5 S x + S gamma5 x, the chirally symmetric form of D_ov^+ D_ov (reading G22).
    With S^2 = 1 it IS gamma5 D gamma5 D; with a polynomial sign of error delta the two differ by 1 - S^2 = O(delta), but
    A' commutes with gamma5 EXACTLY for any Hermitian S and restricted to chirality s it is sector_op: the eigenvectors
    computed per sector are exact eigenvectors of A' whatever delta is, and a chiral source stays in its sector."""
    return 2.0 * x + gamma5(apply_sign(x)) + apply_sign(gamma5(x))


def chirality_of(x: np.ndarray) -> int:
    """+1 / -1 if x has a definite chirality (the other half is exactly zero), else 0."""
    up = np.any(x[..., :2, :] != 0)
    lo = np.any(x[..., 2:, :] != 0)
    return +1 if (up and not lo) else (-1 if (lo and not up) else 0)


def dense_sign(w: np.ndarray, Zv: np.ndarray) -> np.ndarray:
    """sign(H_w) = Z sign(Lambda) Z^+ as a dense matrix (w, Zv from oracle.dense.eig_hw)."""
    return (Zv * np.sign(w)) @ Zv.conj().T


def dense_normal(w: np.ndarray, Zv: np.ndarray) -> np.ndarray:
    """Dense A = (gamma5 + S)^2 from the exact sign."""
    N = Zv.shape[0]
    g5 = np.tile(np.repeat([1.0, 1.0, -1.0, -1.0], 3), N // 12)
    H = np.diag(g5).astype(np.complex128) + dense_sign(w, Zv)
    return H @ H


def dense_sector_modes(A: np.ndarray, s: int, k: int, spinor_shape):
    """The k lowest eigenpairs of A restricted to chirality s, by dense eigendecomposition of the sector block.
    Returns (mu ascending [k], W [k] + spinor_shape with gamma5 W_j = s W_j)."""
    N = A.shape[0]
    g5 = np.tile(np.repeat([1.0, 1.0, -1.0, -1.0], 3), N // 12)
    idx = np.nonzero(g5 == s)[0]
    B = A[np.ix_(idx, idx)]
    mu, Y = np.linalg.eigh(0.5 * (B + B.conj().T))
    W = np.zeros((k, N), dtype=np.complex128)
    W[:, idx] = Y[:, :k].T
    return mu[:k], W.reshape((k,) + tuple(spinor_shape))


def deflated_multishift_cg(apply_A, W, mu, sigmas, b, tol: float, maxiter: int):
    """(A + sigma_i) x_i = b with the eigenpairs (mu_j, W[j]) of A deflated.  Returns (xs, iterations of the CG on the
    projected source, true relative residuals |b - (A + sigma_i) x_i| / |b| with A itself)."""
    shape = b.shape
    bv = b.reshape(-1).astype(np.complex128)
    Wm = np.asarray(W, dtype=np.complex128).reshape(len(mu), -1)
    c = Wm.conj() @ bv                                   # c_j = w_j^+ b
    b_perp = bv - Wm.T @ c
    xs_cg, it, _ = multishift_cg(apply_A, sigmas, b_perp.reshape(shape), tol * np.linalg.norm(bv) / np.linalg.norm(b_perp), maxiter)
    xs, res = [], np.empty(len(sigmas))
    for i, sg in enumerate(sigmas):
        x = xs_cg[i].reshape(-1) + Wm.T @ (c / (np.asarray(mu) + sg))
        xs.append(x.reshape(shape))
        r = bv - (apply_A(x.reshape(shape)).reshape(-1) + sg * x)
        res[i] = np.linalg.norm(r) / np.linalg.norm(bv)
    return xs, it, res
