"""CPU-only tests of the product's host logic and of the C-ABI surface (no compute calls)."""
import ctypes
import re
import os

import numpy as np
import pytest

import paper_1111_6288_b200 as ovp
from paper_1111_6288_b200 import build as ovbuild
from oracle import chebyshev as ch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    ovbuild.build()
    return ovp.load_library()


def test_library_exports_every_declared_symbol(lib):
    hdr = open(os.path.join(ROOT, "include", "ov.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(ov_[a-z0-9_]+)\s*\(", hdr))
    assert declared == set(ovp.SYMBOLS)
    for name in declared:
        assert hasattr(lib, name), name


def test_chebyshev_coeffs_match_oracle_generator(lib):
    for n, se in [(0, 0.3), (1, 0.2), (13, 0.06), (32, 0.05), (200, 0.02), (300, 0.01)]:
        got = ovp.chebyshev_coeffs(n, se * se)
        ref = ch.cheb_coeffs(n, se * se)
        assert np.max(np.abs(got - ref)) <= 1e-12 * np.max(np.abs(ref))
    with pytest.raises(ovp.OvError):
        ovp.chebyshev_coeffs(5, 0.0)


def test_host_eigh_against_numpy(lib):
    rng = np.random.default_rng(0)
    for n in (1, 2, 3, 5, 40, 130, 216):
        A = rng.standard_normal((n, n)) + 1j * rng.standard_normal((n, n))
        A = A + A.conj().T
        w, Z = ovp.host_eigh(A)
        assert np.max(np.abs(w - np.linalg.eigvalsh(A))) < 1e-11 * max(1.0, np.abs(w).max())
        assert np.max(np.abs(Z.conj().T @ Z - np.eye(n))) < 1e-12
        assert np.max(np.abs(A @ Z - Z * w)) < 1e-10 * max(1.0, np.abs(w).max())
    # real symmetric tridiagonal + arrow (the Lanczos projected matrix)
    n = 60
    T = np.diag(rng.standard_normal(n)) + 0j
    for i in range(20, n - 1):
        T[i, i + 1] = T[i + 1, i] = rng.standard_normal()
    T[:20, 20] = rng.standard_normal(20)
    T[20, :20] = T[:20, 20]
    w, Z = ovp.host_eigh(T)
    assert np.max(np.abs(w - np.linalg.eigvalsh(T))) < 1e-12
    assert np.max(np.abs(T @ Z - Z * w)) < 1e-12
    # degenerate spectra (no rotation needed / all equal / repeated) and the size of configs[4]'s Krylov space, which must
    # not stall the GPU for seconds per restart cycle any more (the Jacobi sweeps of rounds 1-2 took 8.9 s here)
    for A in (np.eye(7), np.zeros((6, 6)), np.diag([3.0, 1.0, 2.0, 2.0, -1.0])):
        w, Z = ovp.host_eigh(A.astype(np.complex128))
        assert np.array_equal(w, np.sort(np.diag(A))) and np.max(np.abs(A @ Z - Z * w)) == 0.0
    import time
    n = 416
    A = rng.standard_normal((n, n)) + 1j * rng.standard_normal((n, n))
    A = A + A.conj().T
    t0 = time.perf_counter()
    w, Z = ovp.host_eigh(A)
    assert time.perf_counter() - t0 < 3.0
    assert np.max(np.abs(w - np.linalg.eigvalsh(A))) < 1e-11 * np.abs(w).max()
    assert np.max(np.abs(Z.conj().T @ Z - np.eye(n))) < 1e-12
    assert np.max(np.abs(A @ Z - Z * w)) < 1e-10 * np.abs(w).max()


def test_no_cpu_fallback(lib):
    """Without a CUDA device the product path refuses loudly instead of computing on the host."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("CUDA device present")
    with pytest.raises(ovp.OvError):
        ovp.Overlap((4, 4, 4, 4), 0.19, np.zeros((4, 4, 4, 4, 4, 3, 3), dtype=np.complex128))
    ctx = ctypes.c_void_p()
    dims = (ctypes.c_int * 4)(4, 4, 4, 4)
    rc = lib.ov_create(ctypes.byref(ctx), dims, ctypes.c_double(0.19), ctypes.c_void_p(8), ctypes.c_int(18), None)
    assert rc == ovp.binding.OV_ECUDA and not ctx.value


def test_bench_algorithmic_bytes():
    """bench.py's roofline numerator: per sign, n Clenshaw orders of 2 launches + the final launch."""
    import bench
    V = 1000
    # n = 1: launch 1 (960) + launch 2 (960 + 2 operands, no b_{j+2} yet) + final (960 + x [+ x_low])
    assert bench.algorithmic_bytes_per_sign(1, V, False) == (960 + (960 + 384) + (960 + 192)) * V
    assert bench.algorithmic_bytes_per_sign(1, V, True) == (960 + (960 + 384) + (960 + 384)) * V
    n = 300
    per_site = bench.algorithmic_bytes_per_sign(n, 1, True)
    assert per_site == n * 2496 - 192 + 960 + 384          # 2496 B/site per order
    assert bench.algorithmic_bytes_per_sign(n, 1, True, recon=12) == per_site - (2 * n + 1) * 192
    assert bench.aggregate_value(1, 8, 1000.0) == 8.0


def test_options_struct_matches_header():
    """binding.OvOptions mirrors struct ov_options of include/ov.h field by field (6 ints + 1 double = 32 bytes)."""
    import ctypes
    import re
    from paper_1111_6288_b200.binding import OvOptions
    src = open(os.path.join(ROOT, "include", "ov.h")).read()
    body = re.search(r"typedef struct ov_options \{(.*?)\} ov_options;", src, re.S).group(1)
    body = re.sub(r"/\*.*?\*/", "", body, flags=re.S)
    fields = [(m.group(1), m.group(2)) for m in re.finditer(r"(int|double)\s+(\w+)\s*;", body)]
    ctype = {"int": ctypes.c_int, "double": ctypes.c_double}
    assert [(n, ctype[t]) for t, n in fields] == list(OvOptions._fields_)
    assert ctypes.sizeof(OvOptions) == 32
