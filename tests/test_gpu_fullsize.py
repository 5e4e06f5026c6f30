"""GPU parity at BASELINE.json's full sizes, in the launch configuration bench.py times (default kernel variant,
recon 18): configs[1] (8^3x16, 64 sources), configs[2] (16^3x32, n=200, k=50 from the GPU Lanczos) and the headline
configs[3] (24^3x64, n=300, k=100).  The oracle consumes the GPU's low modes only after checking them with its
own H_w (O9: residual, orthonormality, Rayleigh quotient).  Plus a property that holds at any size: the
free-field plane-wave eigenvalue in closed form at 24^3x64.
"""
import numpy as np
import pytest
import torch

import oracle
import workloads as wl

pytestmark = pytest.mark.gpu

TOL_HW = 1e-12
TOL_DOV = 1e-10


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


def test_config1_64_sources_dslash_and_hw(ovp):
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


def run_dov_config(ovp, cfg, nsrc_checked, lanczos_order=100):
    U = wl.su3_links(cfg.dims, cfg.spread, wl.gauge_seed(cfg.index))
    op = ovp.Overlap(cfg.dims, cfg.kappa, U)
    coef = ovp.chebyshev_coeffs(cfg.order, cfg.eps)
    op.set_polynomial(coef, cfg.eps, cfg.norm)
    V, lam, res, ok = op.lanczos_lowmodes(cfg.k, tol=1e-8, max_restarts=60, cheb_order=lanczos_order)
    assert ok and np.all(res <= 1e-8)
    Vh = host(op, V)
    check_modes_with_oracle(cfg, U, Vh, lam)
    op.set_smallspace(V, lam)
    errs = []
    for j in range(nsrc_checked):
        x = wl.gaussian_source(cfg.dims, wl.source_seed(cfg.index, j))
        got = host(op, op.apply_dov(0.0, dev(op, x)))
        ref = oracle.dov(cfg.dims, cfg.kappa, U, coef, cfg.eps, cfg.norm, Vh, lam, 0.0, x)
        errs.append(rel(got, ref))
        assert errs[-1] <= TOL_DOV
    # the host-buffer entry point (what bench.py's e2e times) gives the same answer as the device entry point
    x = wl.gaussian_source(cfg.dims, wl.source_seed(cfg.index, 0))
    assert rel(op.apply_dov_host(0.0, x), host(op, op.apply_dov(0.0, dev(op, x)))) <= 1e-14
    return errs


def test_config2_dov_with_lanczos_modes(ovp):
    run_dov_config(ovp, wl.CONFIGS[2], nsrc_checked=4)


def test_config3_headline_hw_all_sources_and_dov(ovp):
    cfg = wl.CONFIGS[3]
    U = wl.su3_links(cfg.dims, cfg.spread, wl.gauge_seed(cfg.index))
    op = ovp.Overlap(cfg.dims, cfg.kappa, U)
    for j in range(cfg.nsrc):
        x = wl.gaussian_source(cfg.dims, wl.source_seed(cfg.index, j))
        assert rel(host(op, op.apply_hw(dev(op, x))), oracle.hw(cfg.dims, cfg.kappa, U, x)) <= TOL_HW
    del op
    torch.cuda.empty_cache()
    run_dov_config(ovp, cfg, nsrc_checked=1)


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


@pytest.mark.skipif(not __import__("os").environ.get("OV_LONG_TESTS"),
                    reason="configs[4] (32^3x64, k=200) takes ~10 min of Lanczos and ~115 GB of HBM: set OV_LONG_TESTS=1")
def test_config4_multishift_cg_true_residuals(ovp):
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
    x, iters, relres, okc = op.multishift_cg(cfg.masses, b, tol=1e-8, maxiter=200)
    assert okc and np.all(relres <= 1e-8) and iters > 0
