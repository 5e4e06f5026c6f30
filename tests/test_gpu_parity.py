"""GPU parity tests: the CUDA path (through the C ABI) against the CPU oracle, element by element, on the
same seeded inputs.  Tolerances (BASELINE.json north_star): rel-L2 <= 1e-12 per Wilson apply,
<= 1e-10 per sign / D_ov apply.  Run on the B200 box with  pytest -m gpu.
"""
import numpy as np
import pytest
import torch

import oracle
from oracle import chebyshev as ch
from oracle import dense
from oracle.multishift_cg import multishift_cg, sigma_of_mass
import workloads as wl

pytestmark = pytest.mark.gpu

KAPPA = 0.19
NORM = 1.0 + 8.0 * KAPPA
TOL_HW = 1e-12
TOL_DOV = 1e-10


def rel(a, b):
    return np.linalg.norm((a - b).ravel()) / np.linalg.norm(b.ravel())


@pytest.fixture(scope="module")
def ovp():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_1111_6288_b200 as m
    from paper_1111_6288_b200 import build
    build.build()
    return m


def make(ovp, dims, U, recon=18, variant=0):
    op = ovp.Overlap(dims, KAPPA, U, recon=recon)
    if variant:
        op.set_dslash_variant(variant)
    return op


def to_dev(op, x):
    return op.pack_spinor(torch.from_numpy(np.ascontiguousarray(x)).cuda())


def to_host(op, x):
    return op.unpack_spinor(x).cpu().numpy()


# ------------------------------------------------------------------------------------------ layout
def test_pack_unpack_roundtrip(ovp):
    dims = (4, 2, 6, 8)
    op = make(ovp, dims, wl.unit_links(dims))
    x = np.stack([wl.gaussian_source(dims, s) for s in (1, 2, 3)])
    d = to_dev(op, x)
    assert d.shape == (3, 12, op.V)
    # ABI layout (include/ov.h): V = 384 is a multiple of 32 -> blocked [V/32][12][32]
    assert op.spinor_layout == 1
    ref = x.reshape(3, op.V // 32, 32, 12).transpose(0, 1, 3, 2).reshape(3, 12, op.V)
    assert np.array_equal(d.cpu().numpy(), ref)
    assert np.array_equal(to_host(op, d), x)
    # a volume that is not a multiple of 32 uses planes [12][V]
    dims2 = (6, 6, 2, 2)
    op2 = make(ovp, dims2, wl.unit_links(dims2))
    x2 = wl.gaussian_source(dims2, 4)
    d2 = to_dev(op2, x2)
    assert op2.spinor_layout == 0
    assert np.array_equal(d2.cpu().numpy(), x2.reshape(op2.V, 12).T)
    assert np.array_equal(to_host(op2, d2), x2)


# ------------------------------------------------------------------------------------------ Wilson kernel
@pytest.mark.parametrize("dims,spread", [((4, 4, 4, 4), 0.3), ((4, 2, 6, 8), 0.6), ((8, 8, 8, 16), 0.5),
                                         ((24, 4, 4, 2), 0.8), ((6, 10, 2, 4), 0.4), ((6, 6, 2, 6), 0.5),
                                         ((2, 2, 2, 2), 0.7), ((8, 4, 4, 3), 0.6), ((16, 8, 4, 6), 0.7),
                                         ((8, 12, 8, 5), 0.5), ((8, 4, 4, 2), 0.6), ((24, 8, 12, 4), 0.7),
                                         ((32, 4, 8, 3), 0.5)])
@pytest.mark.parametrize("recon", [18, 12])
def test_dslash_and_hw_vs_oracle(ovp, dims, spread, recon):
    U = wl.su3_links(dims, spread, wl.gauge_seed(1))
    nsrc = 3
    x = np.stack([wl.gaussian_source(dims, wl.source_seed(1, j)) for j in range(nsrc)])
    ref_hop = np.stack([oracle.wilson_hop(dims, U, v) for v in x])
    ref_hw = np.stack([oracle.hw(dims, KAPPA, U, v) for v in x])
    op = make(ovp, dims, U, recon)
    X, Y, Z, T = dims
    tma = X % 8 == 0 and Y % 4 == 0 and Z % 4 == 0         # the shapes the TMA-staged kernel (variant 2) takes
    assert op.dslash_variant == (2 if tma else 1)           # ... and the automatic choice
    results = {}
    for variant in ((1, 2) if tma else (1,)):
        op.set_dslash_variant(variant)
        d = to_dev(op, x)
        hop = to_host(op, torch.stack([op.dslash(d[j]) for j in range(nsrc)]))   # single-rhs launches: the chosen variant
        got = to_host(op, torch.stack([op.apply_hw(d[j]) for j in range(nsrc)]))
        assert rel(hop, ref_hop) <= TOL_HW
        for j in range(nsrc):
            assert rel(got[j], ref_hw[j]) <= TOL_HW
        results[variant] = (hop, got)
        # the batched launch (always the gather kernel) agrees too
        assert rel(to_host(op, op.apply_hw(d)), ref_hw) <= TOL_HW
    if tma:   # same arithmetic in the same order: the hop agrees to the last bit, H_w up to the compiler's FMA contraction
        assert np.array_equal(results[1][0], results[2][0]) and rel(results[1][1], results[2][1]) <= 1e-15
    if not tma:
        with pytest.raises(ovp.OvError):
            op.set_dslash_variant(2)


def test_hw_rejects_aliasing_and_bad_args(ovp):
    dims = (4, 4, 4, 4)
    op = make(ovp, dims, wl.unit_links(dims))
    x = op.new_spinor()
    with pytest.raises(ovp.OvError):
        op.apply_hw(x, out=x)
    with pytest.raises(ovp.OvError):
        op.apply_sign(x)  # no polynomial set
    with pytest.raises(ovp.OvError):
        op.set_polynomial([1.0, 0.5], 0.0, NORM)
    V = op.new_spinor(2)
    op.set_polynomial([1.0, 0.5], 0.01, NORM)
    with pytest.raises(ovp.OvError):
        op.set_smallspace(V, [0.1, 0.0])  # sign(0) undefined


def test_hw_host_entry_point(ovp):
    dims = (4, 2, 6, 8)
    U = wl.su3_links(dims, 0.5, 5)
    x = np.stack([wl.gaussian_source(dims, 6 + j) for j in range(5)])   # 5 rhs: both staging buffers are re-used twice
    op = make(ovp, dims, U)
    ref = np.stack([oracle.hw(dims, KAPPA, U, v) for v in x])
    got = op.apply_hw_host(x)                                            # pageable host memory
    assert rel(got, ref) <= TOL_HW
    xp = torch.from_numpy(x).pin_memory()                                # pinned: H2D / D2H overlap the operator
    outp = torch.empty_like(xp).pin_memory()
    for _ in range(2):                                                   # a second call re-uses the pipeline
        outp.zero_()
        op.apply_hw_host(xp, outp)
        assert rel(outp.numpy(), ref) <= TOL_HW
    op.set_polynomial(ovp.chebyshev_coeffs(6, 0.04), 0.04, NORM)
    gd = op.apply_dov_host(0.1, xp[:3].contiguous().pin_memory())
    for j in range(3):
        assert rel(gd[j].numpy(), oracle.dov(dims, KAPPA, U, ovp.chebyshev_coeffs(6, 0.04), 0.04, NORM, None, None, 0.1, x[j])) <= TOL_DOV


# ------------------------------------------------------------------------------------------ BLAS-1
def test_blas(ovp):
    dims = (6, 10, 2, 4)  # 12*480 = 5760 elements: several warps plus a ragged tail
    op = make(ovp, dims, wl.unit_links(dims))
    x = wl.gaussian_source(dims, 1)
    y = wl.gaussian_source(dims, 2)
    dx, dy = to_dev(op, x), to_dev(op, y)
    d = op.blas_dot(dx, dy)
    assert abs(d - np.vdot(x, y)) <= 1e-13 * np.linalg.norm(x) * np.linalg.norm(y)
    assert abs(op.blas_norm2(dx) - np.vdot(x, x).real) <= 1e-13 * np.vdot(x, x).real
    assert op.blas_dot(dx, dy) == d  # bit-reproducible
    a = 0.3 - 1.7j
    op.blas_axpy(a, dx, dy)
    assert rel(to_host(op, dy), y + a * x) <= 1e-15
    op.blas_scale(-2.5, dx)
    assert rel(to_host(op, dx), -2.5 * x) <= 1e-15


# ------------------------------------------------------------------------------------------ config 0: 4^4
@pytest.fixture(scope="module")
def cfg0():
    cfg = wl.CONFIGS[0]
    U = wl.su3_links(cfg.dims, cfg.spread, wl.gauge_seed(0))
    w, Zv, _, _ = dense.eig_hw(cfg.dims, cfg.kappa, U)
    x = wl.gaussian_source(cfg.dims, wl.source_seed(0, 0))
    V, lam = dense.lowest_modes(w, Zv, cfg.norm, cfg.k, x.shape)
    return dict(cfg=cfg, U=U, w=w, Z=Zv, x=x, V=V, lam=lam)


def setup_op(ovp, c, recon=18, variant=0, with_small=True):
    cfg = c["cfg"]
    op = make(ovp, cfg.dims, c["U"], recon, variant)
    coef = ovp.chebyshev_coeffs(cfg.order, cfg.eps)
    op.set_polynomial(coef, cfg.eps, cfg.norm)
    if with_small:
        op.set_smallspace(to_dev(op, c["V"]), c["lam"])
    return op, coef


def test_projector_vs_numpy(ovp, cfg0):
    op, _ = setup_op(ovp, cfg0)
    x = cfg0["x"]
    V = cfg0["V"].reshape(len(cfg0["lam"]), -1)
    c = V.conj() @ x.ravel()
    perp, low, coef = op.project(to_dev(op, x))
    assert np.max(np.abs(coef - c)) <= 1e-13 * np.linalg.norm(x)
    assert rel(to_host(op, perp), (x.ravel() - c @ V).reshape(x.shape)) <= 1e-13
    assert rel(to_host(op, low), ((np.sign(cfg0["lam"]) * c) @ V).reshape(x.shape)) <= 1e-13


@pytest.mark.parametrize("recon", [18, 12])
@pytest.mark.parametrize("with_small", [True, False])
def test_config0_sign_and_dov(ovp, cfg0, recon, with_small):
    c = cfg0
    cfg = c["cfg"]
    op, coef = setup_op(ovp, c, recon, with_small=with_small)
    V, lam = (c["V"], c["lam"]) if with_small else (None, None)
    x = c["x"]
    dx = to_dev(op, x)
    ref_s = oracle.sign(cfg.dims, cfg.kappa, c["U"], coef, cfg.eps, cfg.norm, V, lam, x)
    assert rel(to_host(op, op.apply_sign(dx)), ref_s) <= TOL_DOV
    for mass in (0.0, 0.1):
        ref_d = oracle.dov(cfg.dims, cfg.kappa, c["U"], coef, cfg.eps, cfg.norm, V, lam, mass, x)
        assert rel(to_host(op, op.apply_dov(mass, dx)), ref_d) <= TOL_DOV
    # and against the exact dense sign, within the polynomial's own error (reading G15)
    exact = dense.exact_sign_apply(c["w"], c["Z"], x)
    assert rel(to_host(op, op.apply_sign(dx)), exact) <= ch.delta_measured(coef, cfg.eps)
    got_host = op.apply_dov_host(0.0, x)
    assert rel(got_host, oracle.dov(cfg.dims, cfg.kappa, c["U"], coef, cfg.eps, cfg.norm, V, lam, 0.0, x)) <= TOL_DOV


def test_degenerate_orders(ovp, cfg0):
    c = cfg0
    cfg = c["cfg"]
    op = make(ovp, cfg.dims, c["U"])
    dx = to_dev(op, c["x"])
    for n in (0, 1, 2):
        coef = ovp.chebyshev_coeffs(n, 0.04)
        op.set_polynomial(coef, 0.04, cfg.norm)
        ref = oracle.sign(cfg.dims, cfg.kappa, c["U"], coef, 0.04, cfg.norm, None, None, c["x"])
        assert rel(to_host(op, op.apply_sign(dx)), ref) <= TOL_DOV


def test_multishift_cg_vs_oracle(ovp, cfg0):
    c = cfg0
    cfg = c["cfg"]
    op, coef = setup_op(ovp, c)
    masses = (0.1, 0.005, 0.04)
    x, iters, res, ok = op.multishift_cg(masses, to_dev(op, c["x"]), tol=1e-9, maxiter=300)
    assert ok and np.all(res <= 1e-8)

    def g5(v):
        o = v.copy(); o[..., 2:, :] *= -1; return o
    args = (cfg.dims, cfg.kappa, c["U"], coef, cfg.eps, cfg.norm, c["V"], c["lam"])
    A = lambda v: g5(oracle.dov(*args, 0.0, g5(oracle.dov(*args, 0.0, v))))
    xs, it_ref, res_ref = multishift_cg(A, [sigma_of_mass(m) for m in masses], c["x"], 1e-9, 300)
    assert abs(iters - it_ref) <= 1
    got = to_host(op, x)
    for i in range(len(masses)):
        assert rel(got[i], xs[i]) <= 1e-7  # two CG runs to tol 1e-9 each


def test_lanczos_4x4_vs_dense(ovp, cfg0):
    c = cfg0
    cfg = c["cfg"]
    op, _ = setup_op(ovp, c, with_small=False)
    k = 8
    V, lam, res, ok = op.lanczos_lowmodes(k, tol=1e-9, max_restarts=40, cheb_order=20, subspace=40)
    assert ok and np.all(res <= 1e-9)
    q = c["w"] / cfg.norm
    exact = q[np.argsort(np.abs(q))[:k]]
    assert np.max(np.abs(np.sort(lam) - np.sort(exact))) <= 1e-9
    Vh = to_host(op, V)
    for i in range(k):  # the oracle's own operator confirms each pair
        r = oracle.hw(cfg.dims, cfg.kappa, c["U"], Vh[i]) / cfg.norm - lam[i] * Vh[i]
        assert np.linalg.norm(r.ravel()) <= 1e-8
    G = Vh.reshape(k, -1).conj() @ Vh.reshape(k, -1).T
    assert np.max(np.abs(G - np.eye(k))) <= 1e-10


# ------------------------------------------------------------------------------------------ T-small on the GPU
def test_small_space_needed_on_gpu(ovp, parity_log):
    """The oracle's pin P11 run through the CUDA path: sqrt(eps) sits between q_k and q_{k+1}, the source lives mostly in
    the k low modes, so without the small space the polynomial alone is wrong at O(1) on them, and with it the result is
    within delta of the exact dense sign -- a wrong sign(lambda_i), a dropped v_i or a mis-ordered coefficient fails here."""
    dims = (4, 4, 4, 4)
    U = wl.su3_links(dims, 0.5, 77)
    w, Zv, _, _ = dense.eig_hw(dims, KAPPA, U)
    q = np.sort(np.abs(w)) / NORM
    k = 10
    se = 0.5 * (q[k - 1] + q[k])
    coef = ch.cheb_coeffs(60, se * se)
    x0 = wl.gaussian_source(dims, 78)
    V, lam = dense.lowest_modes(w, Zv, NORM, k, x0.shape)
    assert (lam > 0).any() and (lam < 0).any()              # both signs present
    x = x0 * 1e-3 + np.tensordot(np.arange(1, k + 1) * (1 + 0.5j), V, axes=(0, 0))
    exact = dense.exact_sign_apply(w, Zv, x)
    d = ch.delta_measured(coef, se * se)
    op = make(ovp, dims, U)
    op.set_polynomial(coef, se * se, NORM)
    dx = to_dev(op, x)
    without = to_host(op, op.apply_sign(dx))
    op.set_smallspace(to_dev(op, V), lam)
    with_k = to_host(op, op.apply_sign(dx))
    e_with, e_without = rel(with_k, exact), rel(without, exact)
    parity_log("4^4 T-small on the GPU: sign with small space vs exact dense sign", e_with, d)
    parity_log("4^4 T-small on the GPU: oracle vs GPU with small space", rel(with_k, oracle.sign(dims, KAPPA, U, coef, se * se, NORM, V, lam, x)), TOL_DOV)
    assert e_with <= d
    assert e_without > 3 * e_with
    assert rel(with_k, oracle.sign(dims, KAPPA, U, coef, se * se, NORM, V, lam, x)) <= TOL_DOV
    assert rel(without, oracle.sign(dims, KAPPA, U, coef, se * se, NORM, None, None, x)) <= TOL_DOV


# ------------------------------------------------------------------------------------------ adaptive CG
def test_reduced_dov_vs_oracle(ovp, cfg0):
    """The truncated series is the oracle's D_ov with the first n'+1 coefficients; the fp32 sweep agrees with the fp64
    one to single-precision rounding (amplified by the Clenshaw recurrence)."""
    c = cfg0
    cfg = c["cfg"]
    op, coef = setup_op(ovp, c)
    dx = to_dev(op, c["x"])
    for n_red in (cfg.order, 20, 7):
        ref = oracle.dov(cfg.dims, cfg.kappa, c["U"], coef[:n_red + 1], cfg.eps, cfg.norm, c["V"], c["lam"], 0.1, c["x"])
        assert rel(to_host(op, op.apply_dov_reduced(0.1, dx, n_red, False)), ref) <= TOL_DOV
        assert rel(to_host(op, op.apply_dov_reduced(0.1, dx, n_red, True)), ref) <= 2e-5
    assert rel(to_host(op, op.apply_dov_reduced(0.0, dx, cfg.order, False)), to_host(op, op.apply_dov(0.0, dx))) <= 1e-14


@pytest.mark.parametrize("mode", [1, 2])
def test_adaptive_multishift_cg(ovp, cfg0, mode):
    c = cfg0
    cfg = c["cfg"]
    op, coef = setup_op(ovp, c)
    masses = (0.1, 0.005, 0.04)
    b = to_dev(op, c["x"])
    x0, it0, res0, ok0 = op.multishift_cg(masses, b, tol=1e-8, maxiter=300)
    op.set_cg_adaptive(mode)
    x1, it1, res1, ok1 = op.multishift_cg(masses, b, tol=1e-8, maxiter=300)
    orders = op.cg_orders()
    op.set_cg_adaptive(0)
    assert ok0 and ok1 and np.all(res1 <= 1e-8)          # true residuals, recomputed with the full fp64 operator
    assert abs(it1 - it0) <= 2
    assert len(orders) == it1 and abs(orders[0]) == cfg.order and min(abs(o) for o in orders) < cfg.order
    if mode == 2:
        assert any(o < 0 for o in orders)                 # some sweeps ran in fp32
    g0, g1 = to_host(op, x0), to_host(op, x1)
    for i in range(len(masses)):
        assert rel(g1[i], g0[i]) <= 1e-6


# ------------------------------------------------------------------------------------------ batched right-hand sides
@pytest.mark.parametrize("with_small", [True, False])
def test_batched_apply_matches_single_and_oracle(ovp, cfg0, with_small):
    """nrhs > 1 goes through batched Wilson launches (2 rhs per block, up to 4 per sweep): same arithmetic per rhs."""
    c = cfg0
    cfg = c["cfg"]
    op, coef = setup_op(ovp, c, with_small=with_small)
    V, lam = (c["V"], c["lam"]) if with_small else (None, None)
    xs = np.stack([wl.gaussian_source(cfg.dims, 50 + j) for j in range(7)])   # 4 + 3: a full and a ragged batch
    d = to_dev(op, xs)
    got_d, got_s, got_h = to_host(op, op.apply_dov(0.05, d)), to_host(op, op.apply_sign(d)), to_host(op, op.apply_hw(d))
    for j in range(len(xs)):
        dj = to_dev(op, xs[j])
        assert np.array_equal(got_d[j], to_host(op, op.apply_dov(0.05, dj)))
        assert np.array_equal(got_s[j], to_host(op, op.apply_sign(dj)))
        assert np.array_equal(got_h[j], to_host(op, op.apply_hw(dj)))
    ref = oracle.dov(cfg.dims, cfg.kappa, c["U"], coef, cfg.eps, cfg.norm, V, lam, 0.05, xs[6])
    assert rel(got_d[6], ref) <= TOL_DOV


def test_batched_gather_sweep_vs_oracle_on_many_blocks(ovp, parity_log):
    """The batched Clenshaw sweep of the GATHER kernel (two right-hand sides per thread block sharing the link loads, fused
    axpy operands with a right-hand-side stride) meets the oracle on a lattice the TMA-staged kernel does not take
    (X = 6) and that spans many thread blocks (2880 sites; 4^4, the other non-TMA test lattice, is 4 blocks), with a
    small space: nrhs = 5 = one batch of 4 and a single.  The low modes come from the library's Lanczos and are
    re-verified with the oracle's H_w before the oracle uses them."""
    dims, spread, n, se, k = (6, 10, 6, 8), 0.5, 24, 0.05, 6
    U = wl.su3_links(dims, spread, 31)
    op = make(ovp, dims, U)
    assert op.dslash_variant == 1 and op.spinor_layout == 1
    coef = ovp.chebyshev_coeffs(n, se * se)
    op.set_polynomial(coef, se * se, NORM)
    V, lam, res, ok = op.lanczos_lowmodes(k, tol=1e-10, max_restarts=80, cheb_order=40)
    assert ok and np.all(res <= 1e-10)
    Vh = to_host(op, V)
    for i in range(k):
        assert np.linalg.norm((oracle.hw(dims, KAPPA, U, Vh[i]) / NORM - lam[i] * Vh[i]).ravel()) <= 1e-9
    op.set_smallspace(V, lam)
    xs = np.stack([wl.gaussian_source(dims, 80 + j) for j in range(5)])
    got_d, got_s = to_host(op, op.apply_dov(0.07, to_dev(op, xs))), to_host(op, op.apply_sign(to_dev(op, xs)))
    for j in (0, 3, 4):                                       # first and last of the batch of 4, and the single
        ref = oracle.dov(dims, KAPPA, U, coef, se * se, NORM, Vh, lam, 0.07, xs[j])
        e = rel(got_d[j], ref)
        parity_log(f"6x10x6x8 batched gather sweep (nrhs=5, k={k}, n={n}): D_ov rel-L2, rhs {j}", e, TOL_DOV)
        assert e <= TOL_DOV
    ref = oracle.sign(dims, KAPPA, U, coef, se * se, NORM, Vh, lam, xs[2])
    assert rel(got_s[2], ref) <= TOL_DOV
    for j in range(5):                                        # and every rhs equals its own nrhs = 1 call bit for bit
        assert np.array_equal(got_d[j], to_host(op, op.apply_dov(0.07, to_dev(op, xs[j]))))


@pytest.mark.parametrize("k", [401, 801])
def test_batched_projector_with_many_modes(ovp, cfg0, k):
    """The batched V^+ x keeps 128 B of shared memory per (mode, rhs): groups of 4 fit up to k = 400, groups of 2 up to 800.
    Beyond that the batch must fall back to smaller groups (k = 401: pairs; k = 801: one at a time) instead of failing,
    with the per-rhs result unchanged.  V: any orthonormal set does for the projector algebra (QR of a Gaussian matrix)."""
    cfg = cfg0["cfg"]
    rng = np.random.default_rng(k)
    n = 12 * wl.volume(cfg.dims)
    Qm, _ = np.linalg.qr(rng.standard_normal((n, k)) + 1j * rng.standard_normal((n, k)))
    V = np.ascontiguousarray(Qm.T).reshape((k,) + cfg0["x"].shape)
    lam = rng.uniform(0.01, 0.05, k) * rng.choice([-1.0, 1.0], k)
    op = make(ovp, cfg.dims, cfg0["U"])
    op.set_polynomial(ovp.chebyshev_coeffs(4, cfg.eps), cfg.eps, cfg.norm)
    op.set_smallspace(to_dev(op, V), lam)
    xs = np.stack([wl.gaussian_source(cfg.dims, 70 + j) for j in range(5)])    # a group of 4 and a single
    got = to_host(op, op.apply_sign(to_dev(op, xs)))
    for j in range(len(xs)):
        assert np.array_equal(got[j], to_host(op, op.apply_sign(to_dev(op, xs[j]))))
    # the low part is exact on span(V): sign(v_0) = sign(lam_0) v_0 up to the polynomial acting on rounding noise
    assert rel(to_host(op, op.apply_sign(to_dev(op, V[0]))), np.sign(lam[0]) * V[0]) <= 1e-12


def test_timing_hooks_and_launch_count(ovp, cfg0):
    """bench.py's roofline reads these: every launch inside the Clenshaw sweep is the Wilson kernel (2n+1 per sign)."""
    op, _ = setup_op(ovp, cfg0)
    dx = to_dev(op, cfg0["x"])
    out = torch.empty_like(dx)
    op.timing_enable(True)
    l0 = op.launch_count
    for _ in range(3):
        op.apply_dov(0.0, dx, out)
    t = op.timing_read()
    op.timing_enable(False)
    n = cfg0["cfg"].order
    assert t["wilson_launches"] == 3 * (2 * n + 1) and t["wilson_ms"] > 0
    assert t["projector_launches"] == 3 * 4 and t["projector_ms"] > 0
    assert op.launch_count - l0 == 3 * (2 * n + 1 + 4 + 1)      # + projector (4) + the b_n = c_n x axpby
    with pytest.raises(ovp.OvError):
        op.set_dslash_variant(2)


# ------------------------------------------------------------------------------------------ TMA-staged kernel in the sweep
@pytest.mark.parametrize("recon", [18, 12])
def test_tma_variant_sign_and_dov_vs_oracle(ovp, recon):
    """The Clenshaw sweep through the TMA-staged kernel (every epilogue form: 0-3 fused axpy operands) on a lattice of
    several pencils and time segments with a ragged slice count, against the oracle and against the gather kernel."""
    dims = (16, 8, 4, 6)
    U = wl.su3_links(dims, 0.6, 91)
    x = wl.gaussian_source(dims, 92)
    se, n = 0.2, 12
    coef = ovp.chebyshev_coeffs(n, se * se)
    rng = np.random.default_rng(93)
    # any orthonormal set serves as a "small space" for parity (both sides get the same V, lambda)
    A = rng.standard_normal((3, x.size)) + 1j * rng.standard_normal((3, x.size))
    Qm, _ = np.linalg.qr(A.T)
    V = np.ascontiguousarray(Qm.T).reshape((3,) + x.shape)
    lam = np.array([0.05, -0.07, 0.11])
    op = make(ovp, dims, U, recon)
    op.set_polynomial(coef, se * se, NORM)
    op.set_smallspace(to_dev(op, V), lam)
    dx = to_dev(op, x)
    ref_s = oracle.sign(dims, KAPPA, U, coef, se * se, NORM, V, lam, x)
    ref_d = oracle.dov(dims, KAPPA, U, coef, se * se, NORM, V, lam, 0.07, x)
    out = {}
    for variant in (2, 1):
        op.set_dslash_variant(variant)
        assert op.dslash_variant == variant
        s, d = to_host(op, op.apply_sign(dx)), to_host(op, op.apply_dov(0.07, dx))
        assert rel(s, ref_s) <= TOL_DOV and rel(d, ref_d) <= TOL_DOV
        out[variant] = (s, d)
    # same arithmetic in the same order; the compiler's FMA contraction may differ between the two kernels
    print(f"  TMA-staged vs gather kernel, recon {recon}: sign {rel(out[1][0], out[2][0]):.3e}, D_ov {rel(out[1][1], out[2][1]):.3e}")
    assert rel(out[1][0], out[2][0]) <= 1e-14 and rel(out[1][1], out[2][1]) <= 1e-14


# ------------------------------------------------------------------------------------------ links that are not SU(3)
def test_fallback_when_tensor_maps_are_unavailable(ovp, monkeypatch):
    """If tensor maps cannot be built (driver entry point missing, encode refused -- forced here with OV_NO_TMA), a context
    in automatic mode must not fail at every Wilson launch: it falls back at ov_create_ex to what a non-eligible lattice
    gets (blocked layout, gather kernel), still matches the oracle, and refuses an explicit variant 2."""
    dims = (8, 4, 4, 6)
    U = wl.su3_links(dims, 0.5, 5)
    x = wl.gaussian_source(dims, 6)
    ref = oracle.hw(dims, KAPPA, U, x)
    op = make(ovp, dims, U)
    assert op.dslash_variant == 2 and op.spinor_layout == 0
    assert rel(to_host(op, op.apply_hw(to_dev(op, x))), ref) <= TOL_HW
    monkeypatch.setenv("OV_NO_TMA", "1")
    op = make(ovp, dims, U)
    assert op.dslash_variant == 1 and op.spinor_layout == 1
    assert rel(to_host(op, op.apply_hw(to_dev(op, x))), ref) <= TOL_HW
    with pytest.raises(ovp.OvError):
        op.set_dslash_variant(2)
    op = ovp.Overlap(dims, KAPPA, U, layout="planes")          # explicit planes layout: kept, but the gather kernel runs
    assert op.dslash_variant == 1 and op.spinor_layout == 0
    assert rel(to_host(op, op.apply_hw(to_dev(op, x))), ref) <= TOL_HW
    monkeypatch.setenv("OV_NO_TMA", "0")                        # "0" does not switch it off
    assert make(ovp, dims, U).dslash_variant == 2


def test_u3_and_dirichlet_links(ovp):
    """recon 18 takes any 3x3 links: a U(1) background phase on every link (U -> e^{-iqA} U) and zero links
    across a Dirichlet boundary in x and t; recon 12 must refuse them (row 2 could not be rebuilt)."""
    dims = (4, 2, 6, 8)
    U = wl.su3_links(dims, 0.6, 31)
    rng = np.random.default_rng(32)
    phase = np.exp(-1j * 0.7 * rng.standard_normal(U.shape[:5]))          # one U(1) phase per link
    Ub = U * phase[..., None, None]
    Ub[:, :, :, -1, 0] = 0.0                                               # no hop across the x boundary
    Ub[-1, :, :, :, 3] = 0.0                                               # nor across the t boundary
    x = wl.gaussian_source(dims, 33)
    op = make(ovp, dims, Ub, recon=18)
    assert rel(to_host(op, op.apply_hw(to_dev(op, x))), oracle.hw(dims, KAPPA, Ub, x)) <= TOL_HW
    with pytest.raises(ovp.OvError):
        make(ovp, dims, Ub, recon=12)
    make(ovp, dims, U, recon=12)                                           # genuine SU(3) links are accepted


@pytest.mark.parametrize("variant", [1, 2])
@pytest.mark.parametrize("t_boundary,bc_t", [("periodic", 1.0), ("open", 0.0), ("antiperiodic", -1.0)])
def test_background_field_and_boundaries_api_vs_oracle(ovp, variant, t_boundary, bc_t):
    """The library's own background field + Dirichlet walls (ov_options: field, wall_mask, t_boundary)
    against the oracle fed with the links of workloads.background_field / the oracle's boundary factors: the two sides
    implement eq. 4.1 and the walls independently.  8^3 x 16 (configs[1] shape), both Wilson kernels, H_w and D_ov."""
    dims = (8, 8, 8, 16)
    qE, fdir, org = 0.0123, 1, 3
    U = wl.su3_links(dims, 0.5, 61)
    x = wl.gaussian_source(dims, 62)
    Uo = wl.background_field(U, dims, qE, fdir, origin=org)              # oracle side: the field as input links
    bc = (1.0, 0.0, 1.0, bc_t)                                           # wall in y (the field direction), t as asked
    op = ovp.Overlap(dims, KAPPA, U, recon=18, t_boundary=t_boundary, walls=(fdir,), field_dir=fdir, field_qE=qE,
                     field_origin=org)
    op.set_dslash_variant(variant)
    se, n = 0.2, 10
    coef = ovp.chebyshev_coeffs(n, se * se)
    op.set_polynomial(coef, se * se, NORM)
    dx = to_dev(op, x)
    with oracle.boundary(bc):
        ref_h = oracle.hw(dims, KAPPA, Uo, x)
        ref_d = oracle.dov(dims, KAPPA, Uo, coef, se * se, NORM, None, None, 0.05, x)
    assert rel(to_host(op, op.apply_hw(dx)), ref_h) <= TOL_HW
    assert rel(to_host(op, op.apply_dov(0.05, dx)), ref_d) <= TOL_DOV
    assert rel(ref_h, oracle.hw(dims, KAPPA, U, x)) > 1e-3               # the field and the walls do matter
    # 12-real links: rows 0-1 carry the field's phase, the kernels multiply the rebuilt third row by det U (phase-tracked
    # reconstruction) -- same operator, both Wilson kernels, and the fp32 instantiation of the gather kernel
    op12 = ovp.Overlap(dims, KAPPA, U, recon=12, t_boundary=t_boundary, walls=(fdir,), field_dir=fdir, field_qE=qE,
                       field_origin=org)
    op12.set_dslash_variant(variant)
    op12.set_polynomial(coef, se * se, NORM)
    d12 = to_dev(op12, x)
    assert rel(to_host(op12, op12.apply_hw(d12)), ref_h) <= TOL_HW
    assert rel(to_host(op12, op12.apply_dov(0.05, d12)), ref_d) <= TOL_DOV
    assert rel(to_host(op12, op12.apply_hw_f32(d12)), ref_h) <= 5e-7


# ------------------------------------------------------------------------------------------ D_ov low modes, deflated CG
def test_dov_lowmodes_and_deflated_cg_4x4_vs_oracle(ovp, parity_log):
    """SURVEY 8f rank 2 on the oracle's hard 4^4 lattice (smooth links, periodic time: 6 near-zero
    modes of D_ov^+ D_ov per chirality sector).  (a) ov_lanczos_dov_lowmodes per sector = the dense eigenpairs of the
    exact A; (b) the deflated multi-mass CG = the oracle's deflated CG (same iterations +-1, solutions) and the dense
    direct solve; (c) deflation cuts the iterations by > 3."""
    from oracle import deflation as dfl
    dims = (4, 4, 4, 4)
    U = wl.su3_links(dims, 0.3, 41)
    bc = (1.0, 1.0, 1.0, 1.0)
    with oracle.boundary(bc):
        w, Zv, _, _ = dense.eig_hw(dims, KAPPA, U)
    A = dfl.dense_normal(w, Zv)
    shape = (4, 4, 4, 4, 4, 3)
    N = A.shape[0]
    se = 0.9 * np.min(np.abs(w)) / NORM                     # the polynomial covers the whole spectrum of Q: no small space
    n = int(np.ceil(np.log(0.41 / 1e-11) / (2.1 * se)))     # delta ~ 1e-11 by eq. 2.2
    coef = ovp.chebyshev_coeffs(n, se * se)
    op = ovp.Overlap(dims, KAPPA, U, t_boundary="periodic")
    op.set_polynomial(coef, se * se, NORM)
    k = 6
    Ws, mus = [], []
    for s in (+1, -1):
        W, mu, res, ok = op.lanczos_dov_lowmodes(s, k, tol=1e-10, max_restarts=60, cheb_order=12, subspace=30)
        assert ok and np.all(res <= 1e-10)
        mu_ref, _ = dfl.dense_sector_modes(A, s, k, shape)
        err = float(np.max(np.abs(np.sort(mu) - mu_ref)))
        parity_log(f"4^4 D_ov low modes, chirality {s:+d}: max |mu_i - dense mu_i| (mu in [{mu_ref[0]:.1e}, {mu_ref[-1]:.1e}])", err, 1e-9)
        assert err <= 1e-9
        Wh = to_host(op, W)
        for i in range(k):                                   # the dense exact operator confirms each pair; chirality
            v = Wh[i].reshape(-1)
            assert np.linalg.norm(A @ v - mu[i] * v) <= 1e-8
            assert rel(dfl.gamma5(Wh[i]), s * Wh[i]) <= 1e-10
        Ws.append(W); mus.append(mu)
    Wd = torch.cat(Ws).contiguous()
    mud = np.concatenate(mus)
    masses = [0.005, 0.02, 0.1]
    sig = [sigma_of_mass(m) for m in masses]
    b = wl.gaussian_source(dims, 43)
    db = to_dev(op, b)
    x_plain, it_plain, res_plain, ok1 = op.multishift_cg(masses, db, tol=1e-9, maxiter=2000)
    op.set_deflation(Wd, mud)
    x_defl, it_defl, res_defl, ok2 = op.multishift_cg(masses, db, tol=1e-9, maxiter=2000)
    op.set_deflation(None, None)
    assert ok1 and ok2 and np.all(res_plain <= 1e-8) and np.all(res_defl <= 1e-8)
    # the oracle's deflated CG with the oracle's own (dense) modes and the oracle's polynomial D_ov
    mu_p, W_p = dfl.dense_sector_modes(A, +1, k, shape)
    mu_m, W_m = dfl.dense_sector_modes(A, -1, k, shape)
    with oracle.boundary(bc):
        args = (dims, KAPPA, U, coef, se * se, NORM, None, None)
        Aor = lambda v: dfl.normal_op(lambda u: oracle.dov(*args, 0.0, u), v)
        xs, it_ref, res_ref = dfl.deflated_multishift_cg(Aor, np.concatenate([W_p, W_m]), np.concatenate([mu_p, mu_m]),
                                                         sig, b, 1e-9, 2000)
    assert abs(it_defl - it_ref) <= 1
    got = to_host(op, x_defl)
    for i, sg in enumerate(sig):
        e1 = rel(got[i], xs[i])
        direct = np.linalg.solve(A + sg * np.eye(N), b.reshape(-1)).reshape(shape)
        e2 = rel(got[i], direct)
        parity_log(f"4^4 deflated multi-mass CG, mass {masses[i]}: vs oracle deflated CG ({it_defl} vs {it_ref} iterations)", e1, 1e-6)
        parity_log(f"4^4 deflated multi-mass CG, mass {masses[i]}: vs dense direct solve with the exact sign", e2, 1e-6)
        assert e1 <= 1e-6 and e2 <= 1e-6
    parity_log(f"4^4 iterations plain / deflated = {it_plain} / {it_defl}: ratio (gate: >= 3, reported as 3/ratio <= 1)",
               3.0 * it_defl / it_plain, 1.0)
    assert it_plain >= 3 * it_defl


# ------------------------------------------------------------------------------------------ degenerate cases
def test_degenerate_inputs(ovp, cfg0):
    c = cfg0
    cfg = c["cfg"]
    op, _ = setup_op(ovp, c)
    zero = torch.zeros_like(to_dev(op, c["x"]))
    # zero source: nothing to solve
    x, iters, res, ok = op.multishift_cg((0.1, 0.02), zero, tol=1e-8, maxiter=50)
    assert ok and iters == 0 and float(x.abs().max()) == 0.0 and np.all(res == 0.0)
    # iteration limit reached: flagged, the last iterate is returned, true residuals are still reported
    x, iters, res, ok = op.multishift_cg((0.1, 0.02), to_dev(op, c["x"]), tol=1e-12, maxiter=2)
    assert not ok and iters == 2 and np.all(np.isfinite(res)) and np.all(res > 1e-12)
    # operators are linear: the zero vector maps to the zero vector, in every entry point
    for y in (op.apply_hw(zero), op.apply_sign(zero), op.apply_dov(0.3, zero), op.dslash(zero)):
        assert float(y.abs().max()) == 0.0
    # bad arguments
    with pytest.raises(ovp.OvError):
        op.lanczos_lowmodes(0)
    with pytest.raises(ovp.OvError):
        op.lanczos_lowmodes(4, subspace=12 * op.V)           # Krylov space as large as the whole space
    with pytest.raises(ovp.OvError):
        op.multishift_cg((2.5,), zero)                       # mass outside (-2, 2)
    with pytest.raises(ovp.OvError):
        op.apply_dov_reduced(0.0, zero, cfg.order + 1, False)
    with pytest.raises(ovp.OvError):
        ovp.Overlap((4, 4, 4, 1), KAPPA, wl.unit_links((4, 4, 4, 1)))   # every extent must be >= 2


def test_deflation_degenerate_inputs(ovp):
    """Edge cases of the deflation row: bad arguments are refused; a source that lies inside the deflation space is solved
    with zero CG iterations, x_i = w (w^+ b)/(mu + sigma_i); clearing the deflation space restores the plain solver."""
    dims = (4, 4, 4, 4)
    U = wl.su3_links(dims, 0.3, 41)
    with oracle.boundary((1.0, 1.0, 1.0, 1.0)):
        w, _, _, _ = dense.eig_hw(dims, KAPPA, U)
    se = 0.9 * np.min(np.abs(w)) / NORM
    # the defect 1 - sign^2 = O(delta) of a sector eigenvector enters x amplified by 1/(mu + sigma) ~ 1e3 here
    # (include/ov.h, ov_set_deflation): delta ~ 1e-13 by eq. 2.2
    n = int(np.ceil(np.log(0.41 / 1e-13) / (2.1 * se)))
    op = ovp.Overlap(dims, KAPPA, U, t_boundary="periodic")
    with pytest.raises(ovp.OvError):
        op.lanczos_dov_lowmodes(+1, 2)                        # no polynomial yet
    op.set_polynomial(ovp.chebyshev_coeffs(n, se * se), se * se, NORM)
    for bad in (dict(chirality=0, k=2), dict(chirality=2, k=2), dict(chirality=1, k=0)):
        with pytest.raises(ovp.OvError):
            op.lanczos_dov_lowmodes(bad["chirality"], bad["k"])
    W, mu, res, ok = op.lanczos_dov_lowmodes(-1, 3, tol=1e-12, max_restarts=80, cheb_order=12, subspace=30)
    assert ok
    with pytest.raises(ovp.OvError):
        op.set_deflation(W, -np.abs(mu) - 1.0)                # D^+ D has no negative eigenvalue
    op.set_deflation(W, mu)
    masses = (0.01, 0.1)
    b = W[1].clone()                                          # a source inside the deflation space
    x, iters, relres, okc = op.multishift_cg(masses, b, tol=1e-8, maxiter=100)
    assert okc and iters == 0 and np.all(relres <= 1e-8)
    bh, xh = to_host(op, b), to_host(op, x)
    for i, m in enumerate(masses):
        assert rel(xh[i], bh / (mu[1] + sigma_of_mass(m))) <= 1e-8
    # preconditions the solver enforces (include/ov.h, ov_set_deflation): no adaptive modes with a deflation space ...
    op.set_cg_adaptive(1)
    with pytest.raises(ovp.OvError) as ei:
        op.multishift_cg(masses, b, tol=1e-8, maxiter=100)
    assert ei.value.code == ovp.binding.OV_ESTATE
    op.set_cg_adaptive(0)
    # ... and no mu_j + sigma_i <= 0: a zero mode with mass 0 would be divided by zero
    op.set_deflation(W, np.array([0.0, mu[1], mu[2]]))
    with pytest.raises(ovp.OvError) as ei:
        op.multishift_cg((0.0, 0.1), b, tol=1e-8, maxiter=100)
    assert ei.value.code == ovp.binding.OV_EINVAL and "singular" in str(ei.value)
    x0, it0, rr0, ok0 = op.multishift_cg(masses, b, tol=1e-8, maxiter=100)     # the same space with masses > 0 is fine
    assert ok0 and it0 == 0 and np.all(np.isfinite(to_host(op, x0)))
    # a new polynomial (or small space) changes the operator: the deflation space is dropped, not left stale
    op.set_deflation(W, mu)
    op.set_polynomial(ovp.chebyshev_coeffs(n, se * se), se * se, NORM)
    _, iters1, relres1, ok1 = op.multishift_cg(masses, b, tol=1e-8, maxiter=500)
    assert ok1 and iters1 > 0 and np.all(relres1 <= 1e-8)
    op.set_deflation(W, mu)
    assert op.multishift_cg(masses, b, tol=1e-8, maxiter=100)[1] == 0
    op.set_deflation(None, None)
    _, iters2, relres2, ok2 = op.multishift_cg(masses, b, tol=1e-8, maxiter=500)
    assert ok2 and iters2 > 0 and np.all(relres2 <= 1e-8)


# ------------------------------------------------------------------------------------------ chirally symmetric CG operator
def test_symmetric_cg_operator_vs_oracle(ovp, cfg0):
    """ov_set_cg_operator(1): A' = 2 + gamma5 S + S gamma5 (reading G22; oracle.deflation.normal_op_sym, pin P18).
    (a) general source: same iterations (+-1) and solutions as the oracle's multi-shift CG on A'; (b) chiral source: the
    solver detects the chirality, every application costs one sign (about half the launches), same solutions as the
    oracle's general A'."""
    from oracle import deflation as dfl
    c = cfg0
    cfg = c["cfg"]
    op, coef = setup_op(ovp, c)
    op.set_cg_operator(1)
    masses = (0.1, 0.02)
    sig = [sigma_of_mass(m) for m in masses]
    S = lambda v: oracle.sign(cfg.dims, cfg.kappa, c["U"], coef, cfg.eps, cfg.norm, c["V"], c["lam"], v)
    Aop = lambda v: dfl.normal_op_sym(S, v)
    launches = {}
    for name, b in (("general", c["x"]), ("chiral", dfl.chiral_project(c["x"], -1))):
        l0 = op.launch_count
        x, iters, res, ok = op.multishift_cg(masses, to_dev(op, b), tol=1e-9, maxiter=300)
        launches[name] = (op.launch_count - l0) / max(1, iters)
        assert ok and np.all(res <= 1e-8)
        assert op.cg_chirality == (0 if name == "general" else -1)
        xs, it_ref, res_ref = multishift_cg(Aop, sig, b, 1e-9, 300)
        assert abs(iters - it_ref) <= 1
        got = to_host(op, x)
        for i in range(len(masses)):
            assert rel(got[i], xs[i]) <= 1e-7
        if name == "chiral":
            assert rel(dfl.gamma5(got[0]), -got[0]) == 0.0          # the solution has kept the chirality exactly
    assert launches["chiral"] < 0.6 * launches["general"]            # one sign per step instead of two
    op.set_cg_adaptive(1)
    with pytest.raises(ovp.OvError):                                 # the adaptive modes belong to the gamma5 D gamma5 D form
        op.multishift_cg(masses, to_dev(op, c["x"]))


def test_symmetric_operator_makes_deflation_exact(ovp, parity_log):
    """With a polynomial of delta ~ 1e-5 the sector eigenvectors are eigenvectors of gamma5 D gamma5 D only to O(delta), and
    that defect, amplified by 1/(mu + sigma) ~ 1e3-1e4, stalls the deflated solve far above tol; for A' they are exact
    and the deflated solve reaches tol (readings G21, G22)."""
    dims = (4, 4, 4, 4)
    U = wl.su3_links(dims, 0.3, 41)
    with oracle.boundary((1.0, 1.0, 1.0, 1.0)):
        w, _, _, _ = dense.eig_hw(dims, KAPPA, U)
    se = 0.9 * np.min(np.abs(w)) / NORM
    n = int(np.ceil(np.log(0.41 / 1e-5) / (2.1 * se)))
    op = ovp.Overlap(dims, KAPPA, U, t_boundary="periodic")
    op.set_polynomial(ovp.chebyshev_coeffs(n, se * se), se * se, NORM)
    Ws, mus = [], []
    for s in (+1, -1):
        W, mu, res, ok = op.lanczos_dov_lowmodes(s, 6, tol=1e-11, max_restarts=80, cheb_order=12, subspace=30)
        assert ok
        Ws.append(W); mus.append(mu)
    op.set_deflation(torch.cat(Ws).contiguous(), np.concatenate(mus))
    b = to_dev(op, wl.gaussian_source(dims, 43))
    masses = (0.005, 0.1)
    out = {}
    for mode in (0, 1):
        op.set_cg_operator(mode)
        _, iters, relres, ok = op.multishift_cg(masses, b, tol=1e-9, maxiter=500)
        out[mode] = (iters, float(relres.max()))
    parity_log(f"4^4 deflated CG, delta ~ 1e-5, gamma5 D gamma5 D form ({out[0][0]} iterations): true residual (stalls, gate is a LOWER bound)",
               1e-7 / out[0][1], 1.0)
    parity_log(f"4^4 deflated CG, delta ~ 1e-5, symmetric form ({out[1][0]} iterations): true residual", out[1][1], 1e-8)
    assert out[0][1] > 1e-7 and out[1][1] <= 1e-8
