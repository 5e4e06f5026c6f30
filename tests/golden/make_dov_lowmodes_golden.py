"""Writes tests/golden/dov_lowmodes_8x8x8x8.txt: the lowest eigenvalues of A = D_ov(0)^+ D_ov(0) in each chirality sector
on an 8^4 lattice with smooth links and periodic time, computed with the ORACLE only (oracle/overlap_oracle.c for H_w and the
polynomial sign, oracle/deflation.py for the sector operator A_s x = 2x + (s + gamma5) sign(H_w) x) and scipy's ARPACK,
independent of the CUDA library.  ov_lanczos_dov_lowmodes is compared with these values in tests/test_gpu_fullsize.py: a
mode skipped below mu_k shows up as a shifted value (readings G20, G13).

Inputs: workloads.su3_links(dims=(8,8,8,8), spread=0.3, seed=workloads.gauge_seed(8)), kappa = 0.19, norm = 1 + 8 kappa,
boundary factors (1,1,1,1).  Polynomial: sqrt(eps) = 0.9 min|lambda(Q)| (min|lambda| from ARPACK on Q^2), order n with
0.41 exp(-2.1 n sqrt(eps)) = 1e-12 (eq. 2.2), Chebyshev coefficients from oracle/chebyshev.py; no small space.
ARPACK runs on B = 4.2 - A_s (which='LA': the wanted low end of A_s becomes the well-separated top end of B).  Each stored
mu is the Rayleigh quotient w^+ A_s w of the ARPACK vector, accepted only if |A_s w - mu w| <= 1e-9 and gamma5 w = s w.

  python tests/golden/make_dov_lowmodes_golden.py [nmodes=10]        (several minutes on 8 cores)
"""
import os
import sys
import time

import numpy as np
from scipy.sparse.linalg import LinearOperator, eigsh

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
import oracle  # noqa: E402
from oracle import chebyshev as ch  # noqa: E402
from oracle import deflation as dfl  # noqa: E402
import workloads as wl  # noqa: E402

DIMS, SPREAD, CONFIG_SEED, KAPPA = (8, 8, 8, 8), 0.3, 8, 0.19
NORM = 1.0 + 8.0 * KAPPA
BC = (1.0, 1.0, 1.0, 1.0)


def main():
    nmodes = int(sys.argv[1]) if len(sys.argv) > 1 else 10
    U = wl.su3_links(DIMS, SPREAD, wl.gauge_seed(CONFIG_SEED))
    X, Y, Z, T = DIMS
    shape = (T, Z, Y, X, 4, 3)
    N = 12 * X * Y * Z * T
    oracle.set_boundary(BC)
    t0 = time.time()

    def q(v):
        return oracle.hw(DIMS, KAPPA, U, v.reshape(shape)).reshape(-1) / NORM

    Q2 = LinearOperator((N, N), matvec=lambda v: q(q(v)), dtype=np.complex128)
    w, _ = eigsh(Q2, k=2, which="SA", tol=1e-10, ncv=40, maxiter=20000,
                 v0=np.random.default_rng(2).standard_normal(N) + 0j)
    qmin = float(np.sqrt(w.min()))
    se = round(0.9 * qmin, 4)
    n = int(np.ceil(np.log(0.41 / 1e-12) / (2.1 * se)))
    coef = ch.cheb_coeffs(n, se * se)
    print(f"min |lambda(Q)| = {qmin:.6f}, sqrt(eps) = {se}, order {n}  ({time.time() - t0:.0f} s)", flush=True)

    def sign(v):
        return oracle.sign_poly(DIMS, KAPPA, U, coef, se * se, NORM, v)

    lines = []
    for s in (+1, -1):
        napply = [0]

        def a_s(v):
            napply[0] += 1
            x = dfl.chiral_project(v.reshape(shape), s)          # ARPACK's vectors drift out of the sector by rounding only
            return dfl.sector_op(sign, s, x).reshape(-1)

        B = LinearOperator((N, N), matvec=lambda v: 4.2 * dfl.chiral_project(v.reshape(shape), s).reshape(-1) - a_s(v),
                           dtype=np.complex128)
        v0 = dfl.chiral_project((np.random.default_rng(3).standard_normal(N) + 0j).reshape(shape), s).reshape(-1)
        th, vec = eigsh(B, k=nmodes, which="LA", tol=1e-12, ncv=6 * nmodes, maxiter=50000, v0=v0)
        mus, res = [], []
        for i in np.argsort(-th):
            wv = dfl.chiral_project(vec[:, i].reshape(shape), s)
            wv = wv / np.linalg.norm(wv.ravel())
            aw = dfl.sector_op(sign, s, wv)
            mu = np.vdot(wv.ravel(), aw.ravel()).real
            mus.append(mu)
            res.append(np.linalg.norm((aw - mu * wv).ravel()))
            assert np.linalg.norm((dfl.gamma5(wv) - s * wv).ravel()) <= 1e-12
        mus, res = np.array(mus), np.array(res)
        print(f"chirality {s:+d}: {napply[0]} applications, mu = {mus}, max residual {res.max():.2e}  ({time.time() - t0:.0f} s)", flush=True)
        assert np.all(res <= 1e-9), res
        assert np.all(np.diff(mus) > 0)
        lines.append((s, mus, res.max()))
    oracle.set_boundary(oracle.BC_DEFAULT)
    out = os.path.join(ROOT, "tests", "golden", "dov_lowmodes_8x8x8x8.txt")
    with open(out, "w") as f:
        f.write("# lowest eigenvalues of A_s = D_ov^+ D_ov restricted to chirality s (ascending), oracle sign + scipy eigsh on 4.2 - A_s\n")
        f.write("# written by tests/golden/make_dov_lowmodes_golden.py (calls only oracle/ and workloads/); PAPER.md:45, :81, DESIGN.md G20\n")
        f.write(f"# dims {DIMS} spread {SPREAD} gauge seed workloads.gauge_seed({CONFIG_SEED}) kappa {KAPPA} norm {NORM} boundary {BC}\n")
        f.write(f"sqrt_eps = {se}\norder = {n}\n")
        for s, mus, rmax in lines:
            f.write(f"# chirality {s:+d}: max residual |A_s w - mu w| = {rmax:.2e}\n")
            for i, mu in enumerate(mus):
                f.write(f"mu_{'p' if s > 0 else 'm'}_{i} = {mu:.15e}\n")
    print(f"wrote {out} in {time.time() - t0:.0f} s")


if __name__ == "__main__":
    main()
