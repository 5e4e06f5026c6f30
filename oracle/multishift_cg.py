"""ORACLE (test infrastructure only): multi-shift ("multi-mass") CG, O8.

Solves (A + sigma_i) x_i = b for all shifts with one Krylov space, A Hermitian positive (semi)definite,
given as a callback.  For the overlap operator A = D_ov(0)^dagger D_ov(0) = gamma5 D_ov gamma5 D_ov and
sigma_i = m_i^2 / (1 - m_i^2/4)  (reading G10; from D(m)^dagger D(m) = (1 - m^2/4) A + m^2 + O(m delta)).

Recurrences (standard shifted-CG, written with the positive step a and the usual CG beta):
  base system = smallest shift sigma_0, relative shifts s_i = sigma_i - sigma_0 >= 0
  x_i = 0, p_i = b, r = b, zeta_i = zeta_i_old = 1, a_old = 1, beta_old = 0
  q = (A + sigma_0) p_0 ;  a = (r,r)/(p_0,q)
  zeta_i_new = zeta_i zeta_i_old a_old / ( a beta_old (zeta_i_old - zeta_i) + zeta_i_old a_old (1 + s_i a) )
  a_i = a zeta_i_new / zeta_i ;  x_i += a_i p_i ;  r -= a q ;  beta = (r,r)_new / (r,r)_old
  p_i = zeta_i_new r + beta (zeta_i_new/zeta_i)^2 p_i
Shifted residual norm = |zeta_i| ||r||; a system is frozen once it is <= tol ||b||; stop when the base
system (slowest) converges.
"""
from __future__ import annotations

import numpy as np


def sigma_of_mass(m: float) -> float:
    return m * m / (1.0 - 0.25 * m * m)


def multishift_cg(apply_A, sigmas, b, tol: float, maxiter: int):
    """Returns (list of x_i in the order of `sigmas`, iterations, true relative residuals)."""
    sig = np.asarray(sigmas, dtype=np.float64)
    order = np.argsort(sig)
    s0 = sig[order[0]]
    s = sig[order] - s0
    ns = len(sig)
    shape = b.shape
    bv = b.reshape(-1).astype(np.complex128)
    x = [np.zeros_like(bv) for _ in range(ns)]
    p = [bv.copy() for _ in range(ns)]
    r = bv.copy()
    zeta = np.ones(ns)
    zeta_old = np.ones(ns)
    active = np.ones(ns, dtype=bool)
    a_old, beta_old = 1.0, 0.0
    rr = np.vdot(r, r).real
    bnorm = np.sqrt(rr)
    it = 0
    while it < maxiter:
        q = apply_A(p[0].reshape(shape)).reshape(-1) + s0 * p[0]
        a = rr / np.vdot(p[0], q).real
        zeta_new = np.empty(ns)
        for i in range(ns):
            zeta_new[i] = (zeta[i] * zeta_old[i] * a_old /
                           (a * beta_old * (zeta_old[i] - zeta[i]) + zeta_old[i] * a_old * (1.0 + s[i] * a)))
        for i in range(ns):
            if active[i]:
                x[i] += (a * zeta_new[i] / zeta[i]) * p[i]
        r -= a * q
        rr_new = np.vdot(r, r).real
        beta = rr_new / rr
        for i in range(ns):
            if active[i]:
                p[i] = zeta_new[i] * r + beta * (zeta_new[i] / zeta[i]) ** 2 * p[i]
        zeta_old, zeta = zeta, zeta_new
        a_old, beta_old, rr = a, beta, rr_new
        it += 1
        for i in range(ns):
            if active[i] and abs(zeta[i]) * np.sqrt(rr) <= tol * bnorm and i > 0:
                active[i] = False
        if np.sqrt(rr) <= tol * bnorm:
            break
    # undo the sort; true residuals with A itself
    xs = [None] * ns
    res = np.empty(ns)
    for pos, i in enumerate(order):
        xs[i] = x[pos].reshape(shape)
        rt = bv - (apply_A(xs[i]).reshape(-1) + sig[i] * x[pos])
        res[i] = np.linalg.norm(rt) / bnorm
    return xs, it, res
