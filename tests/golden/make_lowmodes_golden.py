"""Writes tests/golden/lowmodes_8x8x8x8.txt: the lowest eigenvalues of Q = H_w/norm on an 8^4 lattice, computed with
the ORACLE's H_w only (oracle/overlap_oracle.c) and scipy's ARPACK (eigsh on Q^2, which='SA'), independent of the CUDA
library.  The GPU Lanczos (ov_lanczos_lowmodes, production parameters) is compared with these values in
tests/test_gpu_fullsize.py: a mode skipped below lambda_k shows up as a shifted value (reading G13;
PAPER.md:39 "a small spectrum of Q around zero", :57).

Inputs: workloads.su3_links(dims=(8,8,8,8), spread=0.5, seed=workloads.gauge_seed(7)), kappa = 0.19, norm = 1 + 8 kappa.
Each stored lambda is the Rayleigh quotient v^+ Q v of the ARPACK vector, accepted only if |Q v - lambda v| <= 1e-9.

  python tests/golden/make_lowmodes_golden.py [nmodes=40]        (a few minutes on 8 cores)
"""
import os
import sys
import time

import numpy as np
from scipy.sparse.linalg import LinearOperator, eigsh

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
import oracle  # noqa: E402
import workloads as wl  # noqa: E402

DIMS, SPREAD, CONFIG_SEED, KAPPA = (8, 8, 8, 8), 0.5, 7, 0.19
NORM = 1.0 + 8.0 * KAPPA


def main():
    nmodes = int(sys.argv[1]) if len(sys.argv) > 1 else 40
    U = wl.su3_links(DIMS, SPREAD, wl.gauge_seed(CONFIG_SEED))
    X, Y, Z, T = DIMS
    shape = (T, Z, Y, X, 4, 3)
    N = 12 * X * Y * Z * T

    def q(v):
        return oracle.hw(DIMS, KAPPA, U, v.reshape(shape)).reshape(-1) / NORM

    A = LinearOperator((N, N), matvec=lambda v: q(q(v)), dtype=np.complex128)
    t0 = time.time()
    w, vec = eigsh(A, k=nmodes, which="SA", tol=1e-13, ncv=4 * nmodes, maxiter=50000,
                   v0=np.random.default_rng(1).standard_normal(N) + 0j)
    order = np.argsort(w)
    lam, res = [], []
    for i in order:
        v = vec[:, i] / np.linalg.norm(vec[:, i])
        qv = q(v)
        l = np.vdot(v, qv).real
        lam.append(l)
        res.append(np.linalg.norm(qv - l * v))
    lam, res = np.array(lam), np.array(res)
    assert np.all(res <= 1e-9), res.max()
    assert np.all(np.diff(np.abs(lam)) > 0)
    assert np.max(np.abs(np.abs(lam) - np.sqrt(w[order]))) <= 1e-10
    out = os.path.join(ROOT, "tests", "golden", "lowmodes_8x8x8x8.txt")
    with open(out, "w") as f:
        f.write("# lowest eigenvalues of Q = H_w/norm (signed, sorted by |lambda|), oracle H_w + scipy eigsh on Q^2\n")
        f.write("# written by tests/golden/make_lowmodes_golden.py (calls only oracle/ and workloads/); SURVEY 8c O9/G13, PAPER.md:39, :57\n")
        f.write(f"# dims {DIMS} spread {SPREAD} gauge seed workloads.gauge_seed({CONFIG_SEED}) kappa {KAPPA} norm {NORM}\n")
        f.write(f"# max residual |Q v - lambda v| = {res.max():.2e}\n")
        for l in lam:
            f.write(f"{l:+.15e}\n")
    print(f"wrote {out}: {nmodes} modes in {time.time() - t0:.0f} s, max residual {res.max():.2e}")


if __name__ == "__main__":
    main()
