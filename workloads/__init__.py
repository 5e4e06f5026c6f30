"""Seeded synthetic inputs shared by the oracle tests, the CUDA parity tests and bench.py.

This module holds NO arithmetic of the method (no Wilson operator, no gamma matrices, no
polynomial, no projector). It only draws random numbers with fixed seeds and shapes them like the
paper's workloads (24^3x64 fp64 lattices, SU(3) links, 12-complex spinors).

Canonical array conventions (reading G16):
  gauge   complex128 [T][Z][Y][X][mu=0..3][row][col]   U_mu(x) links x -> x+mu,  mu = x,y,z,t
  spinor  complex128 [T][Z][Y][X][spin=0..3][colour=0..2]
  site index  i = x + X*(y + Y*(z + Z*t))
"""
from .generators import (  # noqa: F401
    CONFIGS,
    DEFLATION,
    DEFLATION_T_BOUNDARY,
    LatticeConfig,
    su3_links,
    unit_links,
    su3_field,
    background_field,
    dirichlet_walls,
    gaussian_source,
    point_source,
    gauge_seed,
    source_seed,
    volume,
)
