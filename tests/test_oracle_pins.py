"""Pins for the oracle (CPU only): the oracle is checked against what the paper and mathematics fix,
never against itself or the CUDA path.  Pin numbers refer to the table in DESIGN.md.
"""
import numpy as np
import pytest

import oracle
from oracle import chebyshev as ch
from oracle import dense
from oracle.multishift_cg import multishift_cg, sigma_of_mass
import workloads as wl

KAPPA = 0.19
NORM = 1.0 + 8.0 * KAPPA


def rel(a, b):
    return np.linalg.norm((a - b).ravel()) / np.linalg.norm(b.ravel())


def vdot(a, b):
    return np.vdot(a.ravel(), b.ravel())


def g5(psi):
    out = psi.copy()
    out[..., 2:, :] *= -1.0
    return out


# ---------------------------------------------------------------- gamma matrices (reading G2)
def test_gamma_algebra():
    g = [oracle.gamma(i) for i in range(5)]
    for mu in range(4):
        assert np.allclose(g[mu], g[mu].conj().T)
        for nu in range(4):
            anti = g[mu] @ g[nu] + g[nu] @ g[mu]
            assert np.allclose(anti, 2.0 * np.eye(4) * (mu == nu))
    assert np.allclose(g[0] @ g[1] @ g[2] @ g[3], g[4])
    assert np.allclose(g[4], np.diag([1, 1, -1, -1]))


# ---------------------------------------------------------------- P1 hermiticity of H_w
@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (4, 2, 6, 8)])
def test_P1_hw_hermitian(dims):
    U = wl.su3_links(dims, 0.6, 1)
    phi = wl.gaussian_source(dims, 2)
    psi = wl.gaussian_source(dims, 3)
    lhs = vdot(phi, oracle.hw(dims, KAPPA, U, psi))
    rhs = vdot(oracle.hw(dims, KAPPA, U, phi), psi)
    assert abs(lhs - rhs) / abs(lhs) < 1e-13


# ---------------------------------------------------------------- P2 free field, closed form
def _momenta(dims):
    X, Y, Z, T = dims
    for nx in range(X):
        for ny in range(Y):
            for nz in range(Z):
                for nt in range(T):
                    yield (2 * np.pi * nx / X, 2 * np.pi * ny / Y, 2 * np.pi * nz / Z,
                           (2 * nt + 1) * np.pi / T)  # antiperiodic in time


def _plane_wave(dims, p, u):
    X, Y, Z, T = dims
    t, z, y, x = np.meshgrid(np.arange(T), np.arange(Z), np.arange(Y), np.arange(X), indexing="ij")
    ph = np.exp(1j * (p[0] * x + p[1] * y + p[2] * z + p[3] * t))
    return ph[..., None, None] * u.reshape(4, 3)


def test_P2_free_spectrum_closed_form():
    dims = (4, 4, 4, 4)
    w, _, _, herm = dense.eig_hw(dims, KAPPA, wl.unit_links(dims))
    assert herm < 1e-14
    expect = []
    for p in _momenta(dims):
        a = 1.0 - 2.0 * KAPPA * sum(np.cos(p))
        b2 = 4.0 * KAPPA ** 2 * sum(np.sin(p) ** 2)
        lam = np.sqrt(a * a + b2)
        expect += [lam] * 6 + [-lam] * 6
    expect = np.sort(np.array(expect))
    assert np.max(np.abs(np.sort(w) - expect)) < 1e-12
    assert abs(np.min(np.abs(w)) - 0.29793) < 1e-5 and abs(np.max(np.abs(w)) - 2.42364) < 1e-5


def test_P2_plane_wave_dw_convention():
    """D_w e^{ipx} u = (a + 2 i kappa sum_mu gamma_mu sin p_mu) u e^{ipx}: pins (1-gamma_mu) forward,
    the boundary phase and the index order on a non-cubic lattice."""
    dims = (4, 2, 6, 8)
    U = wl.unit_links(dims)
    rng = np.random.default_rng(5)
    moms = list(_momenta(dims))
    for p in [moms[1], moms[37], moms[-3]]:
        u = rng.standard_normal(12) + 1j * rng.standard_normal(12)
        psi = _plane_wave(dims, p, u)
        a = 1.0 - 2.0 * KAPPA * sum(np.cos(p))
        M = a * np.eye(4, dtype=complex)
        for mu in range(4):
            M = M + 2j * KAPPA * np.sin(p[mu]) * oracle.gamma(mu)
        Mu = (M @ u.reshape(4, 3)).reshape(12)
        expect = g5(_plane_wave(dims, p, Mu))
        got = oracle.hw(dims, KAPPA, U, psi)
        assert rel(got, expect) < 1e-13


# ---------------------------------------------------------------- P3 gauge covariance
def test_P3_gauge_covariance():
    dims = (4, 2, 6, 4)
    U = wl.su3_links(dims, 0.7, 11)
    g = wl.su3_field(dims, 1.3, 12)
    psi = wl.gaussian_source(dims, 13)
    Ug = np.empty_like(U)
    for mu, axis in enumerate([3, 2, 1, 0]):  # x,y,z,t -> array axes of [T][Z][Y][X]
        g_fwd = np.roll(g, -1, axis=axis)      # g(x + mu)
        Ug[..., mu, :, :] = np.einsum("...ab,...bc,...dc->...ad", g, U[..., mu, :, :], g_fwd.conj())
    psig = np.einsum("...ab,...sb->...sa", g, psi)
    lhs = oracle.hw(dims, KAPPA, Ug, psig)
    rhs = np.einsum("...ab,...sb->...sa", g, oracle.hw(dims, KAPPA, U, psi))
    assert rel(lhs, rhs) < 1e-13


def test_links_are_su3():
    U = wl.su3_links((4, 4, 4, 4), 0.8, 3)
    UU = np.einsum("...ab,...cb->...ac", U, U.conj())
    assert np.max(np.abs(UU - np.eye(3))) < 1e-13
    assert np.max(np.abs(np.linalg.det(U) - 1.0)) < 1e-13


# ---------------------------------------------------------------- P4-P6 polynomial and eq. 2.2
def test_P4_fig1_minimax(golden):
    n = int(golden["fig1_n"]); se = float(golden["fig1_sqrt_eps"]); d = float(golden["fig1_delta"])
    c, E = ch.minimax_coeffs(n, se * se)
    assert abs(ch.delta_measured(c, se * se) - E) < 1e-6
    assert abs(E - d) < 0.01  # caption prints one digit: delta = 0.1
    # the plain interpolant is worse than the minimax, and the minimax is within eq. 2.2's ballpark
    assert ch.delta_measured(ch.cheb_coeffs(n, se * se), se * se) > E
    assert 0.5 < E / ch.delta_formula(n, se) < 2.0


def test_P5_eq22_slope_and_ratio(golden):
    A = float(golden["eq22_A"]); b = float(golden["eq22_b"])
    assert (ch.A_PAPER, ch.B_PAPER) == (A, b)
    for n, se in [(32, 0.05), (200, 0.02), (300, 0.01)]:
        d = ch.delta_measured(ch.cheb_coeffs(n, se * se), se * se)
        assert 0.8 < d / (A * np.exp(-b * n * se)) < 2.5
    se = 0.05
    d1 = ch.delta_measured(ch.cheb_coeffs(32, se * se), se * se)
    d2 = ch.delta_measured(ch.cheb_coeffs(100, se * se), se * se)
    slope = np.log(d1 / d2) / ((100 - 32) * se)
    assert 1.9 < slope < 2.3


def test_P6_order_without_small_space(golden):
    n = ch.order_formula(1e-10, float(golden["lambda_min"]))
    assert 0.5 * float(golden["order_at_1e-10"]) < n < 2.0 * float(golden["order_at_1e-10"])


def test_cheb_coeffs_interpolate():
    """c_0 convention (G5): P = sum c_j T_j reproduces x^-1/2 exactly at the n+1 nodes."""
    n, eps = 20, 0.01
    c = ch.cheb_coeffs(n, eps)
    th = np.pi * (np.arange(n + 1) + 0.5) / (n + 1)
    xk = 0.5 * ((1 - eps) * np.cos(th) + 1 + eps)
    assert np.max(np.abs(ch.poly_eval(c, eps, xk) * np.sqrt(xk) - 1.0)) < 1e-12


def test_P15_memory_arithmetic(golden):
    dims = [int(v) for v in golden["lattice"].split()]
    nbytes = np.prod(dims) * 12 * 16
    assert abs(nbytes / 1e6 - 169.9) < 0.1
    assert 5.5e9 < int(golden["vectors_per_6GB"]) * nbytes < 6.45e9
    assert round(float(golden["hw_eig_cpu_s"]) * float(golden["cpu_cores"]) /
                 (float(golden["hw_eig_gpu_s"]) * float(golden["gpus"]))) in (34, 35)


# ---------------------------------------------------------------- dense 4^4 brute force (config 0)
@pytest.fixture(scope="module")
def cfg0():
    cfg = wl.CONFIGS[0]
    U = wl.su3_links(cfg.dims, cfg.spread, wl.gauge_seed(0))
    w, Zv, H, herm = dense.eig_hw(cfg.dims, cfg.kappa, U)
    assert herm < 1e-13
    x = wl.gaussian_source(cfg.dims, wl.source_seed(0, 0))
    coef = ch.cheb_coeffs(cfg.order, cfg.eps)
    V, lam = dense.lowest_modes(w, Zv, cfg.norm, cfg.k, x.shape)
    return dict(cfg=cfg, U=U, w=w, Z=Zv, x=x, coef=coef, V=V, lam=lam)


def test_norm_bound(cfg0):
    """reading G3: ||H_w|| <= 1 + 8 kappa for unitary links."""
    assert np.max(np.abs(cfg0["w"])) <= NORM


def test_P7_clenshaw_equals_spectral_polynomial(cfg0):
    """Q P(Q^2) x computed by the Clenshaw loop == Z diag(q P(q^2)) Z^dagger x with P evaluated from
    its definition sum c_j cos(j arccos z): pins the recurrence, alpha/beta, 1/norm and c_0."""
    c = cfg0
    cfg = c["cfg"]
    q = c["w"] / cfg.norm
    f = q * ch.poly_eval(c["coef"], cfg.eps, q * q)
    x = c["x"]
    expect = (c["Z"] @ (f * (c["Z"].conj().T @ x.ravel()))).reshape(x.shape)
    got = oracle.sign_poly(cfg.dims, cfg.kappa, c["U"], c["coef"], cfg.eps, cfg.norm, x)
    assert rel(got, expect) < 1e-12


def test_P7_sign_vs_exact_dense(cfg0):
    c = cfg0
    cfg = c["cfg"]
    x = c["x"]
    exact = dense.exact_sign_apply(c["w"], c["Z"], x)
    dmeas = ch.delta_measured(c["coef"], cfg.eps)
    s_k = oracle.sign(cfg.dims, cfg.kappa, c["U"], c["coef"], cfg.eps, cfg.norm, c["V"], c["lam"], x)
    s_0 = oracle.sign(cfg.dims, cfg.kappa, c["U"], c["coef"], cfg.eps, cfg.norm, None, None, x)
    assert rel(s_k, exact) <= dmeas
    assert rel(s_0, exact) <= dmeas          # gapped workload: polynomial valid on the whole spectrum
    assert rel(s_k, s_0) <= dmeas            # P10
    assert rel(s_k, exact) > 1e-6            # it IS an approximation at n = 32


def test_P7_small_space_exact_on_its_modes(cfg0):
    """sign applied to a low mode v_i returns sign(lambda_i) v_i to rounding."""
    c = cfg0
    cfg = c["cfg"]
    for i in (0, 3, 7):
        v = c["V"][i]
        out = oracle.sign(cfg.dims, cfg.kappa, c["U"], c["coef"], cfg.eps, cfg.norm, c["V"], c["lam"], v)
        assert rel(out, np.sign(c["lam"][i]) * v) < 1e-11


def test_P8_sign_squared(cfg0):
    c = cfg0
    cfg = c["cfg"]
    d = ch.delta_measured(c["coef"], cfg.eps)
    S = lambda v: oracle.sign(cfg.dims, cfg.kappa, c["U"], c["coef"], cfg.eps, cfg.norm, c["V"], c["lam"], v)
    assert rel(S(S(c["x"])), c["x"]) <= 2 * d + d * d


def test_P9_ginsparg_wilson_and_P14_mass(cfg0):
    c = cfg0
    cfg = c["cfg"]
    args = (cfg.dims, cfg.kappa, c["U"], c["coef"], cfg.eps, cfg.norm, c["V"], c["lam"])
    D = lambda m, v: oracle.dov(*args, m, v)
    S = lambda v: oracle.sign(*args, v)
    x = c["x"]
    d = ch.delta_measured(c["coef"], cfg.eps)
    # gamma5 D + D gamma5 - D gamma5 D = gamma5 (1 - S^2)   (identically, for Hermitian S)
    lhs = g5(D(0.0, x)) + D(0.0, g5(x)) - D(0.0, g5(D(0.0, x)))
    rhs = g5(x - S(S(x)))
    assert np.linalg.norm((lhs - rhs).ravel()) / np.linalg.norm(x.ravel()) < 1e-13
    assert np.linalg.norm(lhs.ravel()) / np.linalg.norm(x.ravel()) <= 2 * d + d * d
    # D(m)^dag D(m) x - (1 - m^2/4) A x - m^2 x = m (1 - m/2) (1 - S^2) x,  D^dag = gamma5 D gamma5
    m = 0.1
    Ddag = lambda mm, v: g5(D(mm, g5(v)))
    lhs = Ddag(m, D(m, x)) - (1 - m * m / 4) * Ddag(0.0, D(0.0, x)) - m * m * x
    rhs = m * (1 - m / 2) * (x - S(S(x)))
    assert np.linalg.norm((lhs - rhs).ravel()) / np.linalg.norm(x.ravel()) < 1e-13


def test_P13_free_field_dov_plane_wave():
    """On a free-field plane wave H_w^2 = (a^2+b^2), so Q P(Q^2) psi = P(h^2/norm^2)/norm * H_w psi and
    D_ov psi = psi + gamma5 of that: closed form through poly_eval and the plane-wave D_w."""
    dims = (4, 4, 4, 8)
    U = wl.unit_links(dims)
    n, se = 40, 0.1
    coef = ch.cheb_coeffs(n, se * se)
    p = (2 * np.pi / 4, 0.0, 2 * np.pi * 3 / 4, 3 * np.pi / 8)
    rng = np.random.default_rng(9)
    u = rng.standard_normal(12) + 1j * rng.standard_normal(12)
    psi = _plane_wave(dims, p, u)
    a = 1.0 - 2.0 * KAPPA * sum(np.cos(p))
    b2 = 4.0 * KAPPA ** 2 * sum(np.sin(p) ** 2)
    M = a * np.eye(4, dtype=complex)
    for mu in range(4):
        M = M + 2j * KAPPA * np.sin(p[mu]) * oracle.gamma(mu)
    h2 = (a * a + b2) / NORM ** 2
    assert h2 > se * se
    scale = ch.poly_eval(coef, se * se, np.array([h2]))[0] / NORM
    Mu = (M @ u.reshape(4, 3)).reshape(12)            # D_w u ; gamma5 sign = gamma5 gamma5 D_w * scale
    expect = psi + scale * _plane_wave(dims, p, Mu)
    got = oracle.dov(dims, KAPPA, U, coef, se * se, NORM, None, None, 0.0, psi)
    assert rel(got, expect) < 1e-12
    # and P is close to the exact inverse square root there
    assert abs(scale * NORM * np.sqrt(h2) - 1.0) <= ch.delta_measured(coef, se * se)


# ---------------------------------------------------------------- P11 T-small: the small space is needed
def test_P11_small_space_needed():
    dims = (4, 4, 4, 4)
    U = wl.su3_links(dims, 0.5, 77)
    w, Zv, _, _ = dense.eig_hw(dims, KAPPA, U)
    q = np.sort(np.abs(w)) / NORM
    k = 10
    se = 0.5 * (q[k - 1] + q[k])              # sqrt(eps) between q_k and q_{k+1}
    assert q[k] - q[k - 1] > 1e-4
    n = 60
    coef = ch.cheb_coeffs(n, se * se)
    x0 = wl.gaussian_source(dims, 78)
    V, lam = dense.lowest_modes(w, Zv, NORM, k, x0.shape)
    # a source living mostly in the low modes
    x = x0 * 1e-3 + np.tensordot(np.arange(1, k + 1) * (1 + 0.5j), V, axes=(0, 0))
    exact = dense.exact_sign_apply(w, Zv, x)
    d = ch.delta_measured(coef, se * se)
    with_k = oracle.sign(dims, KAPPA, U, coef, se * se, NORM, V, lam, x)
    without = oracle.sign(dims, KAPPA, U, coef, se * se, NORM, None, None, x)
    assert rel(with_k, exact) <= d
    assert rel(without, exact) > 3 * rel(with_k, exact)


# ---------------------------------------------------------------- P12 T-cg and CG on the overlap operator
def test_P12_multishift_cg_ill_conditioned():
    rng = np.random.default_rng(4)
    N = 400
    spec = np.geomspace(1e-3, 4.0, N)
    Qm, _ = np.linalg.qr(rng.standard_normal((N, N)) + 1j * rng.standard_normal((N, N)))
    A = (Qm * spec) @ Qm.conj().T
    b = rng.standard_normal(N) + 1j * rng.standard_normal(N)
    sig = [sigma_of_mass(m) for m in (0.1, 0.005, 0.04, 0.01, 0.07, 0.02)]
    xs, it, res = multishift_cg(lambda v: A @ v, sig, b, 1e-10, 5000)
    assert it < 5000
    for s, xv in zip(sig, xs):
        direct = np.linalg.solve(A + s * np.eye(N), b)
        assert rel(xv, direct) < 1e-7
    assert np.all(res < 1e-8)


def test_multishift_cg_on_overlap(cfg0):
    c = cfg0
    cfg = c["cfg"]
    args = (cfg.dims, cfg.kappa, c["U"], c["coef"], cfg.eps, cfg.norm, c["V"], c["lam"])
    A = lambda v: g5(oracle.dov(*args, 0.0, g5(oracle.dov(*args, 0.0, v))))
    masses = (0.01, 0.1)
    sig = [sigma_of_mass(m) for m in masses]
    xs, it, res = multishift_cg(A, sig, c["x"], 1e-9, 200)
    assert it < 200 and np.all(res < 1e-8)


# ---------------------------------------------------------------- stored low modes of the 8^4 completeness pin
def test_golden_lowmodes_file_is_this_operator():
    """tests/golden/lowmodes_8x8x8x8.txt is written by tests/golden/make_lowmodes_golden.py (oracle H_w + ARPACK, minutes).
    Cheap consistency check that the file belongs to this operator, seed and norm: a plain 150-step Lanczos on Q^2 with
    the oracle's H_w gives Ritz values that bound the spectrum from inside (theta_min >= lambda_1^2, theta_max <= 1) and,
    at the well-separated upper end, has converged; the lower end must sit within the stored cluster."""
    import os
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "lowmodes_8x8x8x8.txt")
    gold = np.array([float(l) for l in open(path) if l.strip() and not l.startswith("#")])
    assert len(gold) == 40 and np.all(np.diff(np.abs(gold)) > 0) and (gold > 0).any() and (gold < 0).any()
    dims = (8, 8, 8, 8)
    U = wl.su3_links(dims, 0.5, wl.gauge_seed(7))
    shape = (8, 8, 8, 8, 4, 3)
    q = lambda v: oracle.hw(dims, KAPPA, U, v.reshape(shape)).reshape(-1) / NORM
    rng = np.random.default_rng(3)
    v = rng.standard_normal(12 * 4096) + 1j * rng.standard_normal(12 * 4096)
    v /= np.linalg.norm(v)
    m = 150
    Vk = np.zeros((m, v.size), dtype=np.complex128)
    al, be = np.zeros(m), np.zeros(m)
    for j in range(m):
        Vk[j] = v
        w = q(q(v))
        al[j] = np.vdot(v, w).real
        w -= Vk[:j + 1].T @ (Vk[:j + 1].conj() @ w)       # full reorthogonalisation
        w -= Vk[:j + 1].T @ (Vk[:j + 1].conj() @ w)
        be[j] = np.linalg.norm(w)
        v = w / be[j]
    Tm = np.diag(al) + np.diag(be[:-1], 1) + np.diag(be[:-1], -1)
    th = np.linalg.eigvalsh(Tm)
    assert th[0] >= gold[0] ** 2 * (1 - 1e-9)             # variational: no Ritz value below the lowest eigenvalue
    assert th[0] <= gold[-1] ** 2                          # ... and the Krylov space has reached the stored cluster
    assert th[-1] <= 1.0                                   # norm = 1 + 8 kappa bounds the spectrum of Q


# ---------------------------------------------------------------- boundary modes and background field
def test_P13_periodic_time_plane_wave():
    """With the t boundary set periodic the free plane waves carry p_t = 2 pi n / T (not (2n+1) pi / T): pins that the
    boundary factor sits on the hop across t = T-1 <-> 0 and nowhere else."""
    dims = (4, 2, 6, 8)
    U = wl.unit_links(dims)
    rng = np.random.default_rng(6)
    p = (2 * np.pi * 1 / 4, 2 * np.pi * 1 / 2, 2 * np.pi * 5 / 6, 2 * np.pi * 3 / 8)
    u = rng.standard_normal(12) + 1j * rng.standard_normal(12)
    psi = _plane_wave(dims, p, u)
    M = (1.0 - 2.0 * KAPPA * sum(np.cos(p))) * np.eye(4, dtype=complex)
    for mu in range(4):
        M = M + 2j * KAPPA * np.sin(p[mu]) * oracle.gamma(mu)
    expect = g5(_plane_wave(dims, p, (M @ u.reshape(4, 3)).reshape(12)))
    with oracle.boundary((1, 1, 1, 1)):
        got = oracle.hw(dims, KAPPA, U, psi)
    assert rel(got, expect) < 1e-13
    assert rel(oracle.hw(dims, KAPPA, U, psi), expect) > 1e-2      # the default (antiperiodic) is back and differs


def test_P14_dirichlet_equals_zero_links_and_is_hermitian():
    """Boundary factor 0 in a direction = periodic operator on links whose wall links are zero (two routes to the same
    operator: the factor in neighbour() vs the generator's zeroed links), and H_w stays Hermitian."""
    dims = (4, 2, 6, 4)
    U = wl.su3_links(dims, 0.6, 21)
    psi = wl.gaussian_source(dims, 22)
    phi = wl.gaussian_source(dims, 23)
    for dirs in [(3,), (1, 3), (0, 2)]:
        bc = [1.0, 1.0, 1.0, -1.0]
        for mu in dirs:
            bc[mu] = 0.0
        with oracle.boundary(bc):
            a = oracle.hw(dims, KAPPA, U, psi)
            lhs = vdot(phi, a)
            rhs = vdot(oracle.hw(dims, KAPPA, U, phi), psi)
        b = oracle.hw(dims, KAPPA, wl.dirichlet_walls(U, dims, dirs), psi)
        assert rel(a, b) < 1e-15
        assert abs(lhs - rhs) / abs(lhs) < 1e-13
        assert rel(a, oracle.hw(dims, KAPPA, U, psi)) > 1e-3


def test_P15_background_field_plaquette_and_gauge_equivalence():
    """Generator pins (eq. 4.1): every (direction, t) plaquette of the field on unit links is exp(-i qE); and with
    Dirichlet walls in `direction` and t the spectrum cannot depend on `origin` (a constant shift of A_t is a pure
    gauge exp(-i qE origin t)): H_w[origin = 2] = g H_w[origin = 0] g^+ with g(t) = exp(i qE origin t)... checked on a vector."""
    dims = (4, 6, 2, 8)
    X, Y, Z, T = dims
    qE, d = 0.37, 1
    B = wl.background_field(wl.unit_links(dims), dims, qE, d)
    Ud, Ut = B[..., d, 0, 0], B[..., 3, 0, 0]                       # [T][Z][Y][X] phases
    ax = 3 - d
    plaq = Ud * np.roll(Ut, -1, axis=ax) * np.conj(np.roll(Ud, -1, axis=0)) * np.conj(Ut)
    interior = [slice(0, T - 1), slice(None), slice(None), slice(None)]
    interior[ax] = slice(0, dims[d] - 1)
    assert np.max(np.abs(plaq[tuple(interior)] - np.exp(-1j * qE))) < 1e-14
    # origin independence under Dirichlet walls
    U = wl.su3_links(dims, 0.5, 31)
    psi = wl.gaussian_source(dims, 32)
    org = 2
    U0 = wl.dirichlet_walls(wl.background_field(U, dims, qE, d, origin=0), dims, (d, 3))
    U2 = wl.dirichlet_walls(wl.background_field(U, dims, qE, d, origin=org), dims, (d, 3))
    t = np.arange(T).reshape(T, 1, 1, 1, 1, 1)
    g = np.exp(-1j * qE * org * t)                                   # psi'(t) = g(t) psi(t)
    with oracle.boundary((1, 0, 1, 0)):
        lhs = oracle.hw(dims, KAPPA, U2, g * psi)
        rhs = g * oracle.hw(dims, KAPPA, U0, psi)
    assert rel(lhs, rhs) < 1e-13


# ---------------------------------------------------------------- low modes of D_ov and deflation
from oracle import deflation as dfl  # noqa: E402


@pytest.fixture(scope="module")
def hard4():
    """4^4, smooth links, PERIODIC time: D_ov has 12 near-zero modes (the lifted p = 0 modes of the free field)."""
    dims = (4, 4, 4, 4)
    U = wl.su3_links(dims, 0.3, 41)
    bc = (1.0, 1.0, 1.0, 1.0)
    with oracle.boundary(bc):
        w, Zv, H, herm = dense.eig_hw(dims, KAPPA, U)
    assert herm < 1e-13
    A = dfl.dense_normal(w, Zv)
    return dict(dims=dims, U=U, bc=bc, w=w, Zv=Zv, A=A, shape=(4, 4, 4, 4, 4, 3))


def test_P16_normal_operator_chirality_structure(hard4):
    """With the exact sign: A = gamma5 D gamma5 D commutes with gamma5; on a chiral vector it equals the one-sign form
    2x + (s + gamma5) S x; its spectrum lies in [0, 4]; the non-zero levels of the two sectors coincide (pairing)."""
    c = hard4
    A, shape = c["A"], c["shape"]
    N = A.shape[0]
    g5 = np.tile(np.repeat([1.0, 1.0, -1.0, -1.0], 3), N // 12)
    assert np.max(np.abs(A * g5[None, :] - g5[:, None] * A)) < 1e-12             # [A, gamma5] = 0
    assert np.max(np.abs(A - A.conj().T)) < 1e-12
    S = dfl.dense_sign(c["w"], c["Zv"])
    x = wl.gaussian_source(c["dims"], 42)

    def dov0(v):                                                                  # D_ov(0) v with the exact sign
        return v + dfl.gamma5((S @ v.reshape(-1)).reshape(shape))

    ref = dfl.normal_op(dov0, x)
    assert rel((A @ x.reshape(-1)).reshape(shape), ref) < 1e-12
    for s in (+1, -1):
        xs = dfl.chiral_project(x, s)
        one_sign = dfl.sector_op(lambda v: (S @ v.reshape(-1)).reshape(shape), s, xs)
        assert rel(one_sign, dfl.normal_op(dov0, xs)) < 1e-12
        assert rel(dfl.gamma5(one_sign), s * one_sign) < 1e-12                    # stays in its sector
    mu_p, _ = dfl.dense_sector_modes(A, +1, N // 2, shape)
    mu_m, _ = dfl.dense_sector_modes(A, -1, N // 2, shape)
    assert mu_p.min() > -1e-12 and mu_p.max() < 4 + 1e-12 and mu_m.min() > -1e-12 and mu_m.max() < 4 + 1e-12
    inner_p = mu_p[(mu_p > 1e-9) & (mu_p < 4 - 1e-9)]
    inner_m = mu_m[(mu_m > 1e-9) & (mu_m < 4 - 1e-9)]
    assert len(inner_p) == len(inner_m) and np.max(np.abs(inner_p - inner_m)) < 1e-10
    assert mu_p[5] < 0.02 and mu_p[6] > 0.3                                       # 6 near-zero modes per sector, then a gap


def test_P17_deflated_multishift_cg_vs_direct_solve(hard4):
    """Deflated multi-mass CG = dense direct solve for every shift; deflating the 6 + 6 near-zero modes cuts the
    iteration count by more than 3 (PAPER.md:45 quotes 3-4 at m_pi ~ 200 MeV)."""
    c = hard4
    A, shape = c["A"], c["shape"]
    N = A.shape[0]
    b = wl.gaussian_source(c["dims"], 43)
    sig = [sigma_of_mass(m) for m in (0.005, 0.02, 0.1)]

    def apply_A(v):
        return (A @ v.reshape(-1)).reshape(shape)

    mu_p, W_p = dfl.dense_sector_modes(A, +1, 6, shape)
    mu_m, W_m = dfl.dense_sector_modes(A, -1, 6, shape)
    W = np.concatenate([W_p, W_m])
    mu = np.concatenate([mu_p, mu_m])
    xs, it_defl, res = dfl.deflated_multishift_cg(apply_A, W, mu, sig, b, 1e-9, 2000)
    _, it_plain, res_plain = multishift_cg(apply_A, sig, b, 1e-9, 2000)
    assert np.all(res <= 1e-8) and np.all(res_plain <= 1e-8)
    for s, x in zip(sig, xs):
        direct = np.linalg.solve(A + s * np.eye(N), b.reshape(-1)).reshape(shape)
        assert rel(x, direct) < 1e-6
    assert it_plain >= 3 * it_defl, (it_plain, it_defl)


def test_P18_chirally_symmetric_normal_operator():
    """A' = 2 + gamma5 S + S gamma5 with a SLOPPY polynomial sign (delta ~ 1e-2): it differs from gamma5 D gamma5 D by
    exactly 1 - S^2 (so by O(delta)), is Hermitian, commutes with gamma5 to rounding, equals the one-sign sector form on a
    chiral vector and keeps a chiral vector in its sector -- none of which needs S^2 = 1."""
    dims = (4, 4, 4, 4)
    U = wl.su3_links(dims, 0.3, 41)
    se, n = 0.07, 20
    coef = ch.cheb_coeffs(n, se * se)
    assert 1e-3 < ch.delta_measured(coef, se * se) < 0.3
    with oracle.boundary((1.0, 1.0, 1.0, 1.0)):
        S = lambda v: oracle.sign_poly(dims, KAPPA, U, coef, se * se, NORM, v)
        x = wl.gaussian_source(dims, 51)
        y = wl.gaussian_source(dims, 52)
        Ax = dfl.normal_op_sym(S, x)
        dov0 = lambda v: v + dfl.gamma5(S(v))
        diff = Ax - dfl.normal_op(dov0, x)
        size = np.linalg.norm(diff.ravel()) / np.linalg.norm(Ax.ravel())
        assert rel(diff, x - S(S(x))) < 1e-12 and 1e-4 < size < 0.3                # = (1 - S^2) x, visibly non-zero
        assert rel(dfl.gamma5(Ax), dfl.normal_op_sym(S, dfl.gamma5(x))) < 1e-13    # [A', gamma5] = 0
        assert abs(vdot(y, Ax) - vdot(dfl.normal_op_sym(S, y), x)) / abs(vdot(y, Ax)) < 1e-13
        for s in (+1, -1):
            xs = dfl.chiral_project(x, s)
            As = dfl.normal_op_sym(S, xs)
            assert rel(As, dfl.sector_op(S, s, xs)) < 1e-13
            assert rel(dfl.gamma5(As), s * As) < 1e-13
            assert dfl.chirality_of(xs) == s
    assert dfl.chirality_of(x) == 0 and dfl.chirality_of(wl.point_source(dims)) == +1
