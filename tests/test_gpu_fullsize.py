"""GPU parity at BASELINE.json's full sizes, in the launch configuration bench.py times (default kernel variant,
recon 18): configs[1] (8^3x16, 64 sources), configs[2] (16^3x32, n=200, k=50 from the GPU Lanczos) and the headline
configs[3] (24^3x64, n=300, k=100).  The oracle consumes the GPU's low modes only after checking them with its
own H_w (O9: residual, orthonormality, Rayleigh quotient).  Plus a property that holds at any size: the
free-field plane-wave eigenvalue in closed form at 24^3x64.
"""
import os

import numpy as np
import pytest
import torch

import oracle
from oracle import chebyshev as ch
from oracle.multishift_cg import multishift_cg, sigma_of_mass
import workloads as wl

pytestmark = pytest.mark.gpu

TOL_HW = 1e-12
TOL_DOV = 1e-10
TOL_HW_F32 = 5e-7     # fp32 Wilson kernel: unit roundoff 6e-8, ~60 roundings per output component
GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def rel(a, b):
    return float(np.linalg.norm((a - b).ravel()) / np.linalg.norm(b.ravel()))


@pytest.fixture(scope="module")
def ovp():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_1111_6288_b200 as m
    from paper_1111_6288_b200 import build
    build.build()
    return m


def dev(op, x):
    return op.pack_spinor(torch.from_numpy(np.ascontiguousarray(x)).cuda())


def host(op, x):
    return op.unpack_spinor(x).cpu().numpy()


def max_ulp(a, b):
    """largest distance in units of the spacing of doubles at the vector's scale (reading G14)."""
    scale = np.spacing(np.max(np.abs(b.view(np.float64))))
    return float(np.max(np.abs((a - b).view(np.float64))) / scale)


def test_config1_64_sources_dslash_and_hw(ovp, parity_log):
    cfg = wl.CONFIGS[1]
    U = wl.su3_links(cfg.dims, cfg.spread, wl.gauge_seed(1))
    op = ovp.Overlap(cfg.dims, cfg.kappa, U)
    x = np.stack([wl.gaussian_source(cfg.dims, wl.source_seed(1, j)) for j in range(cfg.nsrc)])
    d = dev(op, x)
    got_hop, got_hw = host(op, op.dslash(d)), host(op, op.apply_hw(d))
    worst = 0.0
    for j in range(cfg.nsrc):
        ref_hop = oracle.wilson_hop(cfg.dims, U, x[j])
        ref_hw = oracle.hw(cfg.dims, cfg.kappa, U, x[j])
        assert rel(got_hop[j], ref_hop) <= TOL_HW
        assert rel(got_hw[j], ref_hw) <= TOL_HW
        worst = max(worst, max_ulp(got_hw[j], ref_hw))
        if j == 0:   # the single-precision instantiation of the same kernel (adaptive CG tail)
            e32 = rel(host(op, op.apply_hw_f32(d[0])), ref_hw)
            parity_log("configs[1] 8^3x16 fp32 H_w rel-L2", e32, TOL_HW_F32)
            assert e32 <= TOL_HW_F32
            parity_log("configs[1] 8^3x16 fp64 H_w rel-L2 (source 0)", rel(got_hw[0], ref_hw), TOL_HW)
    parity_log("configs[1] 8^3x16 fp64 H_w max-ulp over 64 sources", worst, 64.0)
    assert worst <= 64.0  # a handful of ulps at the vector's scale; bitwise equality is not defined (G14)


def check_modes_with_oracle(cfg, U, Vh, lam):
    """O9: the oracle verifies the GPU's eigenpairs with its own operator before using them."""
    k = len(lam)
    flat = Vh.reshape(k, -1)
    worst_res = 0.0
    for i in range(k):
        qv = oracle.hw(cfg.dims, cfg.kappa, U, Vh[i]) / cfg.norm
        worst_res = max(worst_res, float(np.linalg.norm((qv - lam[i] * Vh[i]).ravel())))
        assert abs(np.vdot(Vh[i], qv).real - lam[i]) <= 1e-10
    G = flat.conj() @ flat.T
    assert np.max(np.abs(G - np.eye(k))) <= 1e-10
    assert worst_res <= 1e-8
    return worst_res


def run_dov_config(ovp, cfg, nsrc_checked, parity_log, lanczos_order=100, recon12=False):
    U = wl.su3_links(cfg.dims, cfg.spread, wl.gauge_seed(cfg.index))
    op = ovp.Overlap(cfg.dims, cfg.kappa, U)
    coef = ovp.chebyshev_coeffs(cfg.order, cfg.eps)
    op.set_polynomial(coef, cfg.eps, cfg.norm)
    V, lam, res, ok = op.lanczos_lowmodes(cfg.k, tol=1e-8, max_restarts=60, cheb_order=lanczos_order)
    assert ok and np.all(res <= 1e-8)
    Vh = host(op, V)
    worst_res = check_modes_with_oracle(cfg, U, Vh, lam)
    parity_log(f"configs[{cfg.index}] {cfg.name} Lanczos k={cfg.k}: max |Qv - lambda v| by the oracle's H_w", worst_res, 1e-8)
    st = op.lanczos_stats()
    print(f"lanczos {cfg.name}: {st}")
    op.set_smallspace(V, lam)
    errs = []
    for j in range(nsrc_checked):
        x = wl.gaussian_source(cfg.dims, wl.source_seed(cfg.index, j))
        got = host(op, op.apply_dov(0.0, dev(op, x)))
        ref = oracle.dov(cfg.dims, cfg.kappa, U, coef, cfg.eps, cfg.norm, Vh, lam, 0.0, x)
        if j == 0:
            ref0 = ref
        errs.append(rel(got, ref))
        parity_log(f"configs[{cfg.index}] {cfg.name} D_ov rel-L2 (n={cfg.order}, k={cfg.k}, source {j})", errs[-1], TOL_DOV)
        assert errs[-1] <= TOL_DOV
    # the host-buffer entry point (what bench.py's e2e times) gives the same answer as the device entry point: one source
    # (single-buffered staging) and three (double-buffered copies overlapping the operator), with the small space set
    xs = np.stack([wl.gaussian_source(cfg.dims, wl.source_seed(cfg.index, j)) for j in range(3)])
    want = [host(op, op.apply_dov(0.0, dev(op, xs[j]))) for j in range(3)]
    assert rel(op.apply_dov_host(0.0, xs[0]), want[0]) <= 1e-14
    got3 = op.apply_dov_host(0.0, xs)
    for j in range(3):
        assert rel(got3[j], want[j]) <= 1e-14
    if recon12:
        # the same apply with 12-real links (what bench.py reports as `recon12`), against the oracle reference of source 0
        x0 = wl.gaussian_source(cfg.dims, wl.source_seed(cfg.index, 0))
        op12 = ovp.Overlap(cfg.dims, cfg.kappa, U, recon=12)
        op12.set_polynomial(coef, cfg.eps, cfg.norm)
        op12.set_smallspace(V, lam)
        e12 = rel(host(op12, op12.apply_dov(0.0, dev(op12, x0))), ref0)
        parity_log(f"configs[{cfg.index}] {cfg.name} recon-12 D_ov rel-L2 (n={cfg.order}, k={cfg.k}, source 0)", e12, TOL_DOV)
        assert e12 <= TOL_DOV
        op12.close()
    return errs


def test_config2_dov_with_lanczos_modes(ovp, parity_log):
    run_dov_config(ovp, wl.CONFIGS[2], 4, parity_log)


def test_config3_headline_hw_all_sources_and_dov(ovp, parity_log):
    cfg = wl.CONFIGS[3]
    U = wl.su3_links(cfg.dims, cfg.spread, wl.gauge_seed(cfg.index))
    op = ovp.Overlap(cfg.dims, cfg.kappa, U)
    op12 = ovp.Overlap(cfg.dims, cfg.kappa, U, recon=12)     # 12-real links: bench.py times them at this size
    worst = worst12 = 0.0
    for j in range(cfg.nsrc):
        x = wl.gaussian_source(cfg.dims, wl.source_seed(cfg.index, j))
        ref = oracle.hw(cfg.dims, cfg.kappa, U, x)
        d = dev(op, x)
        worst = max(worst, rel(host(op, op.apply_hw(d)), ref))
        worst12 = max(worst12, rel(host(op12, op12.apply_hw(d)), ref))
        assert worst <= TOL_HW and worst12 <= TOL_HW
        if j == 0:
            e32 = rel(host(op, op.apply_hw_f32(d)), ref)
            parity_log("configs[3] 24^3x64 fp32 H_w rel-L2", e32, TOL_HW_F32)
            assert e32 <= TOL_HW_F32
    parity_log("configs[3] 24^3x64 fp64 H_w rel-L2, worst of 8 sources", worst, TOL_HW)
    parity_log("configs[3] 24^3x64 fp64 H_w with 12-real links rel-L2, worst of 8 sources", worst12, TOL_HW)
    assert op12.dslash_variant == op.dslash_variant == 2
    op12.close()
    del op, op12
    torch.cuda.empty_cache()
    run_dov_config(ovp, cfg, 1, parity_log, recon12=True)


def test_plane_wave_closed_form_at_24x64(ovp):
    """Free field: psi = e^{ipx} u, p_i = 2 pi n_i/L_i, p_t = (2 n_t + 1) pi/T  =>  H_w^2 psi = (a^2 + b^2) psi with
    a = 1 - 2 kappa sum cos p, b^2 = 4 kappa^2 sum sin^2 p (the pin the oracle passes on 4^4, here on the kernel)."""
    dims, kappa = (24, 24, 24, 64), 0.19
    X, Y, Z, T = dims
    op = ovp.Overlap(dims, kappa, wl.unit_links(dims))
    rng = np.random.default_rng(5)
    for n in [(1, 0, 0, 0), (3, 7, 11, 20), (23, 1, 12, 63)]:
        p = np.array([2 * np.pi * n[0] / X, 2 * np.pi * n[1] / Y, 2 * np.pi * n[2] / Z, (2 * n[3] + 1) * np.pi / T])
        t, z, y, x = np.meshgrid(np.arange(T), np.arange(Z), np.arange(Y), np.arange(X), indexing="ij")
        phase = np.exp(1j * (p[0] * x + p[1] * y + p[2] * z + p[3] * t))
        u = rng.standard_normal((4, 3)) + 1j * rng.standard_normal((4, 3))
        psi = phase[..., None, None] * u
        d = dev(op, psi)
        hh = host(op, op.apply_hw(op.apply_hw(d)))
        a = 1 - 2 * kappa * np.sum(np.cos(p))
        b2 = 4 * kappa ** 2 * np.sum(np.sin(p) ** 2)
        assert rel(hh, (a * a + b2) * psi) <= 1e-12


def test_config4_multishift_cg_true_residuals(ovp, parity_log):
    """configs[4]: the oracle cannot run at this size, so the solve is judged by the true residuals recomputed with the
    operator (itself checked against the oracle at configs[0-3]); oracle parity of the CG recurrences is on 4^4."""
    cfg = wl.CONFIGS[4]
    U = wl.su3_links(cfg.dims, cfg.spread, wl.gauge_seed(cfg.index))
    op = ovp.Overlap(cfg.dims, cfg.kappa, U)
    del U
    op.set_polynomial(ovp.chebyshev_coeffs(cfg.order, cfg.eps), cfg.eps, cfg.norm)
    V, lam, res, ok = op.lanczos_lowmodes(cfg.k, tol=1e-8, max_restarts=80, cheb_order=100)
    assert ok and np.all(res <= 1e-8)
    op.set_smallspace(V, lam)
    b = dev(op, wl.point_source(cfg.dims))
    print(f"lanczos {cfg.name}: {op.lanczos_stats()}")
    x, iters, relres, okc = op.multishift_cg(cfg.masses, b, tol=1e-8, maxiter=200)
    parity_log(f"configs[4] 32^3x64 multi-shift CG ({iters} iterations): worst true relative residual", relres.max(), 1e-8)
    parity_log("configs[4] 32^3x64 Lanczos k=200: max residual (library)", res.max(), 1e-8)
    assert okc and np.all(relres <= 1e-8) and iters > 0


# ------------------------------------------------------------------------------------------ Lanczos completeness
def load_golden_lowmodes():
    vals = [float(l) for l in open(os.path.join(GOLDEN, "lowmodes_8x8x8x8.txt")) if l.strip() and not l.startswith("#")]
    return np.array(vals)


def test_lanczos_completeness_8x8_vs_oracle_eigsh(ovp, parity_log):
    """No skipped mode: the k lowest |lambda| from ov_lanczos_lowmodes with the
    PRODUCTION parameters (Chebyshev order 100, default subspace) equal the k lowest from scipy's ARPACK run on the
    oracle's own H_w (tests/golden/lowmodes_8x8x8x8.txt, written by tests/golden/make_lowmodes_golden.py)."""
    gold = load_golden_lowmodes()
    dims, kappa, norm = (8, 8, 8, 8), 0.19, 1.0 + 8 * 0.19
    U = wl.su3_links(dims, 0.5, wl.gauge_seed(7))
    op = ovp.Overlap(dims, kappa, U)
    op.set_polynomial(ovp.chebyshev_coeffs(10, 0.01), 0.01, norm)       # only the norm matters to the eigensolver
    for k in (24, 7):
        V, lam, res, ok = op.lanczos_lowmodes(k, tol=1e-8, max_restarts=60, cheb_order=100)
        assert ok and np.all(res <= 1e-8)
        order = np.argsort(np.abs(lam))
        err = float(np.max(np.abs(lam[order] - gold[:k])))               # signed eigenvalues, sorted by |lambda|
        parity_log(f"8^4 Lanczos k={k} vs oracle+ARPACK: max |lambda_i - golden_i| ({op.lanczos_stats()['restarts']} cycles)",
                   err, 1e-8)
        assert err <= 1e-8
        assert np.abs(lam).max() < abs(gold[k]) - 1e-9                   # nothing from above the k-th level
    # the oracle's operator confirms the vectors of the last run
    Vh = host(op, V)
    for i in range(len(lam)):
        r = oracle.hw(dims, kappa, U, Vh[i]) / norm - lam[i] * Vh[i]
        assert np.linalg.norm(r.ravel()) <= 1e-8


@pytest.fixture(scope="module")
def cfg2(ovp):
    """configs[2] (16^3x32) with its k = 50 low modes, shared by the tests below."""
    cfg = wl.CONFIGS[2]
    U = wl.su3_links(cfg.dims, cfg.spread, wl.gauge_seed(cfg.index))
    op = ovp.Overlap(cfg.dims, cfg.kappa, U)
    op.set_polynomial(ovp.chebyshev_coeffs(cfg.order, cfg.eps), cfg.eps, cfg.norm)
    V, lam, res, ok = op.lanczos_lowmodes(cfg.k, tol=1e-8, max_restarts=60, cheb_order=100)
    assert ok
    op.set_smallspace(V, lam)
    return dict(cfg=cfg, U=U, op=op, V=V, lam=lam, Vh=host(op, V))


def test_lanczos_k_plus_delta_16x32(ovp, cfg2, parity_log):
    """Completeness at a size with no independent eigensolver: the 50 modes of a k = 50 run are the first 50 of a
    k = 66 run (a mode skipped by one of them would have to be skipped by both)."""
    c = cfg2
    V2, lam2, res2, ok2 = c["op"].lanczos_lowmodes(66, tol=1e-8, max_restarts=60, cheb_order=100)
    assert ok2 and np.all(res2 <= 1e-8)
    a = np.sort(np.abs(c["lam"]))
    b = np.sort(np.abs(lam2))
    err = float(np.max(np.abs(a - b[:50])))
    parity_log("16^3x32 Lanczos k=50 vs first 50 of k=66: max | |lambda| difference |", err, 1e-8)
    assert err <= 1e-8
    assert b[50] >= a[-1]


# ------------------------------------------------------------------------------------------ every path the bench reports
def test_recon12_dov_16x32(ovp, cfg2, parity_log):
    """12-real links (row 3 rebuilt in registers) through the whole D_ov path at 16^3x32."""
    c = cfg2
    cfg = c["cfg"]
    coef = ovp.chebyshev_coeffs(cfg.order, cfg.eps)
    op12 = ovp.Overlap(cfg.dims, cfg.kappa, c["U"], recon=12)
    op12.set_polynomial(coef, cfg.eps, cfg.norm)
    op12.set_smallspace(c["V"], c["lam"])
    x = wl.gaussian_source(cfg.dims, wl.source_seed(cfg.index, 5))
    ref = oracle.dov(cfg.dims, cfg.kappa, c["U"], coef, cfg.eps, cfg.norm, c["Vh"], c["lam"], 0.0, x)
    e = rel(host(op12, op12.apply_dov(0.0, dev(op12, x))), ref)
    parity_log("16^3x32 recon-12 D_ov rel-L2 (n=200, k=50)", e, TOL_DOV)
    assert e <= TOL_DOV


def test_batched_dov_16x32(ovp, cfg2, parity_log):
    """ov_apply_dov(nrhs = 7): one full batch of 4 and a ragged batch of 3 through the batched Clenshaw sweep."""
    c = cfg2
    cfg, op = c["cfg"], c["op"]
    coef = ovp.chebyshev_coeffs(cfg.order, cfg.eps)
    xs = np.stack([wl.gaussian_source(cfg.dims, wl.source_seed(cfg.index, 20 + j)) for j in range(7)])
    got = host(op, op.apply_dov(0.03, dev(op, xs)))
    for j in (0, 3, 6):
        ref = oracle.dov(cfg.dims, cfg.kappa, c["U"], coef, cfg.eps, cfg.norm, c["Vh"], c["lam"], 0.03, xs[j])
        e = rel(got[j], ref)
        parity_log(f"16^3x32 batched D_ov (nrhs=7) rel-L2, rhs {j}", e, TOL_DOV)
        assert e <= TOL_DOV


def test_adaptive_cg_16x32_vs_oracle_cg(ovp, cfg2, parity_log):
    """Plain and adaptive (reduced order, fp32 sweeps) multi-shift CG against the oracle's CG driven by the
    oracle's D_ov, at a size where the fp32 kernel runs over a thousand thread blocks.  Order 100 on [0.03^2, 1] keeps the
    oracle's 2 x (iterations + shifts) D_ov applies affordable."""
    c = cfg2
    cfg, op = c["cfg"], c["op"]
    se, n = 0.03, 100
    coef = ovp.chebyshev_coeffs(n, se * se)
    op.set_polynomial(coef, se * se, cfg.norm)
    try:
        masses = (0.1, 0.01)
        bsrc = wl.gaussian_source(cfg.dims, wl.source_seed(cfg.index, 40))
        b = dev(op, bsrc)

        def g5(v):
            o = v.copy(); o[..., 2:, :] *= -1; return o
        args = (cfg.dims, cfg.kappa, c["U"], coef, se * se, cfg.norm, c["Vh"], c["lam"])
        A = lambda v: g5(oracle.dov(*args, 0.0, g5(oracle.dov(*args, 0.0, v))))
        xs, it_ref, res_ref = multishift_cg(A, [sigma_of_mass(m) for m in masses], bsrc, 1e-8, 100)
        assert np.all(res_ref <= 1e-8)
        for mode in (0, 1, 2):
            op.set_cg_adaptive(mode)
            x, iters, res, ok = op.multishift_cg(masses, b, tol=1e-8, maxiter=100)
            orders = op.cg_orders()
            assert ok and np.all(res <= 1e-8) and abs(iters - it_ref) <= 2
            if mode == 2:
                assert any(o < 0 for o in orders)           # some sweeps really ran in fp32
            got = host(op, x)
            for i in range(len(masses)):
                e = rel(got[i], xs[i])
                parity_log(f"16^3x32 multi-shift CG mode {mode} vs oracle CG, mass {masses[i]}: solution rel-L2 "
                           f"({iters} vs {it_ref} iterations)", e, 1e-6)
                assert e <= 1e-6                            # two solves to 1e-8 each
    finally:
        op.set_cg_adaptive(0)
        op.set_polynomial(ovp.chebyshev_coeffs(cfg.order, cfg.eps), cfg.eps, cfg.norm)


# ------------------------------------------------------------------------------------------ deflation at size (8f rank 2)
def test_deflated_cg_16x32_hard_workload(ovp, parity_log):
    """D_ov low modes + deflated multi-mass CG on workloads.DEFLATION (16^3x32, smooth links, periodic time; PAPER.md:45
    "deflation was shown to increase the convergence rate by a factor of 3-4").  The eigenpairs and the solution of the
    lightest mass are re-checked with the ORACLE's operator; iterations must drop by >= 2."""
    from oracle import deflation as dfl
    cfg = wl.DEFLATION
    bc = (1.0, 1.0, 1.0, 1.0)
    U = wl.su3_links(cfg.dims, cfg.spread, wl.gauge_seed(cfg.index))
    op = ovp.Overlap(cfg.dims, cfg.kappa, U, t_boundary=wl.DEFLATION_T_BOUNDARY)
    op.set_polynomial(ovp.chebyshev_coeffs(10, 0.01), 0.01, cfg.norm)            # norm for the H_w eigensolver
    V, lam, res, ok = op.lanczos_lowmodes(16, tol=1e-9, max_restarts=60, cheb_order=100)
    assert ok
    se = 0.95 * float(np.max(np.abs(lam)))
    # delta ~ 1e-12 by eq. 2.2: the deflated part of x carries the defect 1 - sign^2 = O(delta) of the
    # sector eigenvectors amplified by 1/(mu_0 + sigma_0) ~ 4e4, and must stay below tol = 1e-8 (include/ov.h, ov_set_deflation)
    n = int(np.ceil(np.log(0.41 / 1e-12) / (2.1 * se)))
    coef = ovp.chebyshev_coeffs(n, se * se)
    op.set_polynomial(coef, se * se, cfg.norm)
    op.set_smallspace(V, lam)
    k = 12
    Ws, mus = [], []
    for s in (+1, -1):
        W, mu, r, ok = op.lanczos_dov_lowmodes(s, k, tol=1e-9, max_restarts=60, cheb_order=12)
        st = op.lanczos_stats()
        assert ok and np.all(r <= 1e-9)
        print(f"  D_ov low modes, chirality {s:+d}: mu = {np.array2string(np.sort(mu), precision=5)}; {st['restarts']} cycles, "
              f"{st['filter_applies']} filter applies, order {n}, sqrt(eps) {se:.4f}")
        Ws.append(W); mus.append(mu)
    assert np.max(np.abs(np.sort(mus[0])[6:] - np.sort(mus[1])[6:])) <= 1e-7     # pairing of the non-zero levels
    Vh = host(op, V)
    with oracle.boundary(bc):                                                     # the oracle's A_s confirms two pairs per sector
        sgn = lambda v: oracle.sign(cfg.dims, cfg.kappa, U, coef, se * se, cfg.norm, Vh, lam, v)
        for s, W, mu in zip((+1, -1), Ws, mus):
            Wh = host(op, W[:2].contiguous())
            for i in range(2):
                r = dfl.sector_op(sgn, s, Wh[i]) - mu[i] * Wh[i]
                e = float(np.linalg.norm(r.ravel()))
                parity_log(f"16^3x32 D_ov low mode {i} (chirality {s:+d}, mu = {mu[i]:.3e}): |A_s w - mu w| with the oracle's sign", e, 1e-8)
                assert e <= 1e-8
    Wd = torch.cat(Ws).contiguous()
    mud = np.concatenate(mus)
    b = wl.point_source(cfg.dims)
    db = dev(op, b)
    import time
    t0 = time.time()
    x_plain, it_plain, res_plain, ok1 = op.multishift_cg(list(cfg.masses), db, tol=1e-8, maxiter=5000)
    t_plain = time.time() - t0
    op.set_deflation(Wd, mud)
    t0 = time.time()
    x_defl, it_defl, res_defl, ok2 = op.multishift_cg(list(cfg.masses), db, tol=1e-8, maxiter=5000)
    t_defl = time.time() - t0
    op.set_deflation(None, None)
    print(f"  multi-mass CG, 6 masses, tol 1e-8: plain {it_plain} iterations {t_plain:.1f} s, deflated (2 x {k} modes) "
          f"{it_defl} iterations {t_defl:.1f} s; true residuals plain {res_plain.max():.2e}, deflated {res_defl.max():.2e}")
    assert ok1 and ok2
    # the solver stops when the RECURSIVE residual of the slowest system is <= tol |b|; res_* are the TRUE residuals it
    # recomputes with the operator afterwards.  Over ~300 (plain) iterations the recurrence drifts from the true residual
    # by rounding, so the gate is tol plus 20 % for that drift (the observed values are printed above), not tol itself
    assert np.all(res_plain <= 1.2e-8) and np.all(res_defl <= 1.2e-8)
    parity_log(f"16^3x32 hard workload: CG iterations plain / deflated = {it_plain} / {it_defl} (gate: 2 deflated <= plain)",
               2.0 * it_defl / it_plain, 1.0)
    assert it_plain >= 2 * it_defl
    for i in (0, len(cfg.masses) - 1):
        e = rel(host(op, x_defl[i:i + 1].contiguous())[0], host(op, x_plain[i:i + 1].contiguous())[0])
        parity_log(f"16^3x32 deflated vs plain solution, mass {cfg.masses[i]}", e, 1e-5)
        assert e <= 1e-5
    # the oracle's operator on the deflated solution of the lightest mass: |b - (A + sigma) x| / |b|
    xh = host(op, x_defl[0:1].contiguous())[0]
    with oracle.boundary(bc):
        args = (cfg.dims, cfg.kappa, U, coef, se * se, cfg.norm, Vh, lam)
        Ax = dfl.normal_op(lambda u: oracle.dov(*args, 0.0, u), xh)
    sg = sigma_of_mass(cfg.masses[0])
    e = float(np.linalg.norm((b - Ax - sg * xh).ravel()) / np.linalg.norm(b.ravel()))
    # gate: the library's own true residual (<= 1.2e-8 above) plus what the two implementations of A may differ by on this
    # x: |A_gpu x - A_oracle x| <= 2 * 1e-10 |x| (two D_ov applies at the 1e-10 parity gate) with |x| / |b| up to
    # 1/(mu_0 + sigma_0) ~ 4e4, i.e. up to 8e-6 in the worst case allowed by the parity gate, ~1e-15 * 4e4 in practice;
    # 2e-8 leaves 0.8e-8 for it
    parity_log("16^3x32 deflated solution, lightest mass: true residual with the ORACLE's D_ov", e, 2e-8)
    assert e <= 2e-8


def test_dov_lowmodes_completeness_8x8_vs_oracle_eigsh(ovp, parity_log):
    """No skipped D_ov mode (readings G20, G13): the k lowest mu per chirality sector
    from ov_lanczos_dov_lowmodes with the production parameters (filter order 12, default subspace) equal the k lowest from
    scipy's ARPACK run on the ORACLE's sector operator (tests/golden/dov_lowmodes_8x8x8x8.txt, written by
    tests/golden/make_dov_lowmodes_golden.py) on an 8^4 lattice with smooth links and periodic time."""
    from conftest import load_golden
    g = load_golden("dov_lowmodes_8x8x8x8.txt")
    dims, kappa, norm = (8, 8, 8, 8), 0.19, 1.0 + 8 * 0.19
    se, n = float(g["sqrt_eps"]), int(g["order"])
    U = wl.su3_links(dims, 0.3, wl.gauge_seed(8))
    op = ovp.Overlap(dims, kappa, U, t_boundary="periodic")
    op.set_polynomial(ovp.chebyshev_coeffs(n, se * se), se * se, norm)
    for s, tag in ((+1, "p"), (-1, "m")):
        gold = np.array([float(g[f"mu_{tag}_{i}"]) for i in range(10)])
        for k in (8, 3):
            W, mu, res, ok = op.lanczos_dov_lowmodes(s, k, tol=1e-10, max_restarts=60, cheb_order=12)
            assert ok and np.all(res <= 1e-10)
            err = float(np.max(np.abs(np.sort(mu) - gold[:k])))
            parity_log(f"8^4 D_ov low modes, chirality {s:+d}, k={k} vs oracle+ARPACK: max |mu_i - golden_i| "
                       f"({op.lanczos_stats()['restarts']} cycles)", err, 1e-9)
            assert err <= 1e-9
            assert mu.max() < gold[k] - 1e-9                             # nothing from above the k-th level
