"""ORACLE (test infrastructure only): the polynomial P(x) ~ x^(-1/2) of PAPER.md:31 and its error.

The paper gives the form  sign(H_w) ~ Q P(Q^2),  P(x) = p_0 + ... + p_n x^n ~ x^(-1/2), the
error measure  delta = |1 - sqrt(x) P(x)|  on the large space and the empirical law
delta = A exp(-b n sqrt(eps)), A = 0.41, b = 2.1 (eq. 2.2).  It does not say how P is
built (readings G4, G5): here P is expanded in Chebyshev polynomials T_j of
z = (2x - 1 - eps)/(1 - eps) on [eps, 1]; the stored c_0 is the true T_0 coefficient, P = sum_j c_j T_j(z).
Two generators:
  cheb_coeffs     plain Chebyshev interpolation of x^(-1/2) at the n+1 first-kind nodes (the default)
  minimax_coeffs  Remez exchange for min max |1 - sqrt(x) P(x)|  (pins the Fig. 1 example)
"""
from __future__ import annotations

import numpy as np

A_PAPER = 0.41
B_PAPER = 2.1


def delta_formula(n: int, sqrt_eps: float) -> float:
    """eq. 2.2: delta = A exp(-b n sqrt(eps))."""
    return A_PAPER * np.exp(-B_PAPER * n * sqrt_eps)


def order_formula(delta: float, sqrt_eps: float) -> float:
    """eq. 2.2 solved for n."""
    return np.log(A_PAPER / delta) / (B_PAPER * sqrt_eps)


def x_to_z(x, eps):
    return (2.0 * np.asarray(x, dtype=np.float64) - 1.0 - eps) / (1.0 - eps)


def cheb_coeffs(n: int, eps: float) -> np.ndarray:
    """DESIGN.md O5: c_j = (2/(n+1)) sum_k f(x_k) cos(j pi (k+1/2)/(n+1)), f = x^(-1/2),
    z_k = cos(pi (k+1/2)/(n+1)), x_k = ((1-eps) z_k + 1 + eps)/2 ; the j = 0 value is halved so that
    c_0 is the true T_0 coefficient."""
    k = np.arange(n + 1, dtype=np.float64)
    theta = np.pi * (k + 0.5) / (n + 1)
    xk = 0.5 * ((1.0 - eps) * np.cos(theta) + 1.0 + eps)
    fk = 1.0 / np.sqrt(xk)
    j = np.arange(n + 1, dtype=np.float64)[:, None]
    c = (2.0 / (n + 1)) * (np.cos(j * theta[None, :]) @ fk)
    c[0] *= 0.5
    return c


def poly_eval(coef, eps: float, x) -> np.ndarray:
    """P(x) = sum_j c_j T_j(z(x)) with T_j(z) = cos(j arccos z) (the definition, not Clenshaw)."""
    z = np.clip(x_to_z(x, eps), -1.0, 1.0)
    th = np.arccos(z)
    j = np.arange(len(coef), dtype=np.float64)
    return np.cos(np.multiply.outer(th, j)) @ np.asarray(coef, dtype=np.float64)


def error_grid(eps: float, npts: int = 20001) -> np.ndarray:
    """Points of [eps,1], Chebyshev-clustered at both ends (the error peaks at x = eps)."""
    th = np.linspace(0.0, np.pi, npts)
    return 0.5 * ((1.0 - eps) * np.cos(th)[::-1] + 1.0 + eps)


def delta_measured(coef, eps: float, npts: int = 20001) -> float:
    """max over [eps,1] of |1 - sqrt(x) P(x)|."""
    x = error_grid(eps, npts)
    return float(np.max(np.abs(1.0 - np.sqrt(x) * poly_eval(coef, eps, x))))


def minimax_coeffs(n: int, eps: float, npts: int = 40001, iters: int = 60):
    """Remez exchange on a fine grid for  min_P max_{[eps,1]} |1 - sqrt(x) P(x)|,  deg P = n.
    Basis phi_j(x) = sqrt(x) T_j(z(x)); unknowns c_0..c_n and the level E; n+2 reference points.
    Returns (coefficients in the T_j basis, levelled error E)."""
    x = error_grid(eps, npts)
    th = np.arccos(np.clip(x_to_z(x, eps), -1.0, 1.0))
    j = np.arange(n + 1, dtype=np.float64)
    Phi = np.sqrt(x)[:, None] * np.cos(np.multiply.outer(th, j))
    # start from the extrema of T_{n+1} mapped to [eps,1]
    ref = np.unique(np.round((npts - 1) * (np.arange(n + 2) / (n + 1.0))).astype(int))
    ref = np.searchsorted(x, 0.5 * ((1 - eps) * np.cos(np.pi * np.arange(n + 2)[::-1] / (n + 1)) + 1 + eps))
    ref = np.clip(ref, 0, npts - 1)
    c = None
    E = 0.0
    for _ in range(iters):
        sgn = (-1.0) ** np.arange(n + 2)
        M = np.concatenate([Phi[ref], sgn[:, None]], axis=1)
        sol = np.linalg.solve(M, np.ones(n + 2))
        c, E = sol[:-1], sol[-1]
        err = 1.0 - Phi @ c
        # new reference: one extremum of err per sign-alternating segment
        s = np.sign(err)
        s[s == 0] = 1
        bounds = np.flatnonzero(np.diff(s)) + 1
        segs = np.split(np.arange(npts), bounds)
        ext = np.array([seg[np.argmax(np.abs(err[seg]))] for seg in segs])
        if len(ext) < n + 2:
            break
        while len(ext) > n + 2:  # drop the smaller end point
            if abs(err[ext[0]]) < abs(err[ext[-1]]):
                ext = ext[1:]
            else:
                ext = ext[:-1]
        if np.array_equal(ext, ref):
            break
        ref = ext
        if np.max(np.abs(err)) - abs(E) < 1e-12 * abs(E):
            break
    return c, abs(float(E))
