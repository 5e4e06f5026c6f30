"""Seeded input generators (links, sources) and the BASELINE.json config table.

No arithmetic of the method lives here; see the package docstring for array conventions.
Recipe:
  links   for every time slice t (in order), draw re then im of A[z][y][x][mu][3][3] ~ N(0,1) from
          numpy.random.default_rng(seed); H = (A + A^dagger)/2 - tr(.)/3; U = exp(i * spread * H)
          (by Hermitian eigendecomposition of H), so U is in SU(3) to rounding.
  sources re then im of psi[t][z][y][x][spin][colour] ~ N(0,1), one rng per source seed.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Tuple

import numpy as np


def volume(dims) -> int:
    X, Y, Z, T = dims
    return int(X) * int(Y) * int(Z) * int(T)


def _exp_i_hermitian(H: np.ndarray, spread: float) -> np.ndarray:
    """exp(i*spread*H) for a batch of Hermitian 3x3 matrices."""
    w, Z = np.linalg.eigh(H)
    ph = np.exp(1j * spread * w)
    return np.einsum("...ik,...k,...jk->...ij", Z, ph, Z.conj())


def _traceless_hermitian(rng: np.random.Generator, shape) -> np.ndarray:
    re = rng.standard_normal(shape + (3, 3))
    im = rng.standard_normal(shape + (3, 3))
    A = re + 1j * im
    H = 0.5 * (A + np.conj(np.swapaxes(A, -1, -2)))
    tr = np.trace(H, axis1=-2, axis2=-1) / 3.0
    H = H - tr[..., None, None] * np.eye(3)
    return H


def su3_links(dims, spread: float, seed: int) -> np.ndarray:
    """Random SU(3) gauge field, complex128 [T][Z][Y][X][4][3][3]."""
    X, Y, Z, T = (int(d) for d in dims)
    rng = np.random.default_rng(seed)
    U = np.empty((T, Z, Y, X, 4, 3, 3), dtype=np.complex128)
    for t in range(T):
        H = _traceless_hermitian(rng, (Z, Y, X, 4))
        U[t] = _exp_i_hermitian(H, spread)
    return U


def su3_field(dims, spread: float, seed: int) -> np.ndarray:
    """One random SU(3) matrix per site (a gauge transformation), complex128 [T][Z][Y][X][3][3]."""
    X, Y, Z, T = (int(d) for d in dims)
    rng = np.random.default_rng(seed)
    g = np.empty((T, Z, Y, X, 3, 3), dtype=np.complex128)
    for t in range(T):
        H = _traceless_hermitian(rng, (Z, Y, X))
        g[t] = _exp_i_hermitian(H, spread)
    return g


def unit_links(dims) -> np.ndarray:
    """Free field: every link is the 3x3 identity."""
    X, Y, Z, T = (int(d) for d in dims)
    U = np.zeros((T, Z, Y, X, 4, 3, 3), dtype=np.complex128)
    U[..., 0, 0] = 1.0
    U[..., 1, 1] = 1.0
    U[..., 2, 2] = 1.0
    return U


def background_field(U: np.ndarray, dims, qE: float, direction: int, origin: int = 0) -> np.ndarray:
    """Constant electric field of strength E along `direction` (0, 1, 2 = x, y, z) for a quark of charge q, as input
    links (eq. 4.1: U_mu -> exp(-i q A_mu) U_mu).  Gauge taken here (the paper does not fix it):
    A_t(x) = E (x_direction - origin), all other components zero, i.e. only the t links get the phase
    exp(-i qE (x_direction - origin)); every (direction, t) plaquette then carries exp(-i qE).  Returns a new array;
    the links are U(3), not SU(3).  Meant to be used with Dirichlet walls in `direction` and t (dirichlet_walls)."""
    X, Y, Z, T = (int(d) for d in dims)
    if direction not in (0, 1, 2):
        raise ValueError("direction must be 0, 1 or 2")
    out = np.array(U, dtype=np.complex128, copy=True)
    coord = np.arange((X, Y, Z)[direction], dtype=np.float64) - float(origin)
    shape = [1, 1, 1, 1]                     # [T][Z][Y][X]
    shape[3 - direction] = coord.size
    phase = np.exp(-1j * float(qE) * coord).reshape(shape)
    out[..., 3, :, :] *= phase[..., None, None]
    return out


def dirichlet_walls(U: np.ndarray, dims, directions) -> np.ndarray:
    """Links with Dirichlet walls: the links that cross the lattice boundary in each of `directions`
    (U_mu at coordinate d_mu - 1) are set to zero, so no hop connects coordinate d_mu - 1 and 0."""
    out = np.array(U, dtype=np.complex128, copy=True)
    for mu in directions:
        idx = [slice(None)] * 4              # [T][Z][Y][X]
        idx[3 - int(mu)] = -1
        out[tuple(idx) + (int(mu),)] = 0.0
    return out


def gaussian_source(dims, seed: int) -> np.ndarray:
    """Gaussian random spinor, complex128 [T][Z][Y][X][4][3], re then im drawn N(0,1)."""
    X, Y, Z, T = (int(d) for d in dims)
    rng = np.random.default_rng(seed)
    re = rng.standard_normal((T, Z, Y, X, 4, 3))
    im = rng.standard_normal((T, Z, Y, X, 4, 3))
    return re + 1j * im


def point_source(dims, site: int = 0, spin: int = 0, colour: int = 0) -> np.ndarray:
    X, Y, Z, T = (int(d) for d in dims)
    psi = np.zeros((T, Z, Y, X, 4, 3), dtype=np.complex128)
    psi.reshape(-1, 4, 3)[site, spin, colour] = 1.0
    return psi


def gauge_seed(config: int) -> int:
    return 11116288 + int(config)


def source_seed(config: int, j: int) -> int:
    return 1000 * int(config) + int(j)


@dataclass(frozen=True)
class LatticeConfig:
    """One row of BASELINE.json `configs` (index = position in that list)."""

    index: int
    dims: Tuple[int, int, int, int]  # X, Y, Z, T
    spread: float
    kappa: float = 0.19
    order: int = 0          # Chebyshev order n of P (degree in x = Q^2); 0 = no polynomial
    sqrt_eps: float = 0.0
    k: int = 0              # small-space modes
    nsrc: int = 1
    masses: Tuple[float, ...] = field(default_factory=tuple)
    name: str = ""

    @property
    def norm(self) -> float:
        # rigorous bound ||H_w|| <= 1 + 8 kappa for unitary links (reading G3)
        return 1.0 + 8.0 * self.kappa

    @property
    def eps(self) -> float:
        return self.sqrt_eps ** 2

    @property
    def sites(self) -> int:
        return volume(self.dims)


CONFIGS = (
    LatticeConfig(0, (4, 4, 4, 4), 0.3, order=32, sqrt_eps=0.05, k=8, nsrc=1, name="4^4"),
    LatticeConfig(1, (8, 8, 8, 16), 0.5, nsrc=64, name="8^3x16"),
    LatticeConfig(2, (16, 16, 16, 32), 0.7, order=200, sqrt_eps=0.02, k=50, nsrc=16, name="16^3x32"),
    LatticeConfig(3, (24, 24, 24, 64), 0.8, order=300, sqrt_eps=0.01, k=100, nsrc=8, name="24^3x64"),
    LatticeConfig(4, (32, 32, 32, 64), 0.8, order=300, sqrt_eps=0.01, k=200, nsrc=1,
                  masses=(0.005, 0.01, 0.02, 0.04, 0.07, 0.1), name="32^3x64"),
)


# The workload of the deflation row: the random links of CONFIGS give D_ov^+ D_ov a
# spectrum in [2.7, 4] (nothing to deflate), so this one is SMOOTH (small spread) and PERIODIC in time: the p = 0 modes of
# the free overlap operator survive as 6 near-zero modes of D_ov^+ D_ov per chirality sector (condition number ~ 1e4-1e5
# at the lightest mass), followed by the p = 2 pi / T shell -- the situation deflation is for.
DEFLATION = LatticeConfig(5, (16, 16, 16, 32), 0.3, masses=(0.005, 0.01, 0.02, 0.04, 0.07, 0.1), name="16^3x32 smooth links, periodic t")
DEFLATION_T_BOUNDARY = "periodic"
