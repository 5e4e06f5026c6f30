"""ORACLE -- TEST INFRASTRUCTURE ONLY (not the product path).

Plain fp64 CPU statement of the hot path of arXiv 1111.6288 (applying D_ov = 1 + gamma5 sign(H_w),
PAPER.md:29-39), used to judge the CUDA library.  Shares no code with paper_1111_6288_b200/.
Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs import this.

  overlap_oracle.c   H_w, Clenshaw polynomial sign, small-space split, D_ov     (C, loops over sites)
  chebyshev.py       coefficients of P(x) ~ x^(-1/2) on [eps,1]; delta; eq. 2.2  (numpy)
  dense.py           dense H_w on tiny lattices, exact sign by eigendecomposition (numpy)
  multishift_cg.py   multi-shift CG on D_ov^dagger D_ov, step by step            (numpy)
  deflation.py       D_ov^dagger D_ov per chirality sector, dense low modes, deflated multi-shift CG (numpy)

Pins: tests/test_oracle_pins.py (see the table in DESIGN.md).  Every function here has a pin.  What the GPU tests cannot
check with it is completeness of the CUDA eigensolvers above 8^4 (H_w: tests/golden/lowmodes_8x8x8x8.txt; D_ov:
tests/golden/dov_lowmodes_8x8x8x8.txt): on larger lattices eigenpairs are verified one by one, see DESIGN.md section 3.
"""
from .capi import (  # noqa: F401
    build,
    gamma,
    wilson_hop,
    hw,
    sign_poly,
    sign,
    dov,
    num_threads,
    set_boundary,
    boundary,
    BC_DEFAULT,
)
