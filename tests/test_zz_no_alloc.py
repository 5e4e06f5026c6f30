"""ov_blas_dot_static: the scalar product for callers that cannot allocate device memory.

Some programs that use this library cannot call cudaMalloc while they run: a lattice code that has handed all of HBM to
its own pool (the eigenvector sets are 17-80 GB, nothing is left over and the call fails), or one that keeps other
streams busy, which cudaMalloc/cudaFree would stall.  ov_blas_dot is closed to them, because its partial-sum buffer
comes from cudaMalloc.  ov_blas_dot_static keeps the partial sums in a fixed 512 KiB array inside libov.so instead (at
most 33 554 432 complex elements) and allocates nothing.  This test checks it against ov_blas_dot, the existing path,
on the same vectors, within the tolerance tests/test_gpu_parity.py::test_blas uses for dot products (1e-13 |x| |y|).

Each case makes two calls in a row: the array is shared and keeps what the previous call wrote, so the second call --
different vectors, and in one case a shorter vector after a longer one -- would show stale partial sums leaking in.

The file sorts last on purpose (pytest -x stops at the first failure; a failure here must not hide other tests).  It
keeps no state from other test files, so it passes alone in a fresh process as well as after the rest of the suite.
"""
import ctypes

import numpy as np
import pytest
import torch

import workloads as wl

pytestmark = pytest.mark.gpu

KAPPA = 0.19
TOL_DOT = 1e-13  # as test_gpu_parity.py::test_blas: |dot - reference| <= 1e-13 |x| |y|


@pytest.fixture(scope="module")
def ovp():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_1111_6288_b200 as m
    from paper_1111_6288_b200 import build
    build.build()
    return m


def _vectors(op, dims, seeds):
    xs = [wl.gaussian_source(dims, s) for s in seeds]
    return xs, [op.pack_spinor(torch.from_numpy(np.ascontiguousarray(x)).cuda()) for x in xs]


def _static_dot(ovp, dx, dy, out):
    ovp.blas_dot_static(dx, dy, out)          # no host synchronisation inside
    torch.cuda.synchronize()
    re, im = out.cpu().tolist()
    return complex(re, im)


# 12*240 = 2880 elements: two full 1024-element blocks and a ragged third; 12*8192 = 98304: 96 blocks
@pytest.mark.parametrize("dims", [(6, 4, 2, 5), (8, 8, 8, 16)])
def test_static_dot_matches_allocating_dot_two_calls(ovp, dims):
    op = ovp.Overlap(dims, KAPPA, wl.unit_links(dims))
    (x, y, z), (dx, dy, dz) = _vectors(op, dims, (11, 12, 13))
    out = torch.full((2,), float("nan"), dtype=torch.float64, device="cuda")   # the caller's output buffer
    # first call: <x, y>; second call straight after it: <z, x> (other data through the same scratch array)
    for (a, b, da, db) in ((x, y, dx, dy), (z, x, dz, dx)):
        want = op.blas_dot(da, db)            # the existing path (scratch from cudaMalloc)
        got = _static_dot(ovp, da, db, out)
        scale = np.linalg.norm(a) * np.linalg.norm(b)
        assert abs(got - want) <= TOL_DOT * scale
        assert abs(got - np.vdot(a, b)) <= TOL_DOT * scale
    # x == y (norm^2) through the same pointer
    got = _static_dot(ovp, dx, dx, out)
    assert abs(got - op.blas_norm2(dx)) <= TOL_DOT * np.linalg.norm(x) ** 2


def test_static_dot_short_call_after_long_call(ovp):
    """A long vector first, then a short one: the partial sums the long call left beyond the short call's range must not
    be read.  Also n = 0 (nothing launched but the final reduction) gives exactly 0."""
    big, small = (8, 8, 8, 16), (6, 4, 2, 5)
    op_b = ovp.Overlap(big, KAPPA, wl.unit_links(big))
    op_s = ovp.Overlap(small, KAPPA, wl.unit_links(small))
    (xb, yb), (dxb, dyb) = _vectors(op_b, big, (21, 22))
    (xs, ys), (dxs, dys) = _vectors(op_s, small, (23, 24))
    out = torch.zeros(1, dtype=torch.complex128, device="cuda")               # 1 complex128 is accepted too
    ovp.blas_dot_static(dxb, dyb, out)
    ovp.blas_dot_static(dxs, dys, out)        # back to back on the same stream: ordered, no race
    torch.cuda.synchronize()
    got = complex(out.cpu().item())
    assert abs(got - op_s.blas_dot(dxs, dys)) <= TOL_DOT * np.linalg.norm(xs) * np.linalg.norm(ys)
    rc = ovp.load_library().ov_blas_dot_static(ctypes.c_void_p(dxs.data_ptr()), ctypes.c_void_p(dys.data_ptr()),
                                               ctypes.c_longlong(0), ctypes.c_void_p(out.data_ptr()), None)
    torch.cuda.synchronize()
    assert rc == ovp.binding.OV_OK and complex(out.cpu().item()) == 0.0


def test_static_dot_rejects_what_does_not_fit(ovp):
    """Beyond the fixed array the call refuses (OV_EINVAL, a message naming the limit) and launches nothing: `out` keeps
    its value.  The pointers are small valid buffers; they are never dereferenced."""
    lib = ovp.load_library()
    nmax = ovp.blas_dot_static_max()
    assert nmax == 32768 * 1024
    buf = torch.ones(4, dtype=torch.complex128, device="cuda")
    out = torch.full((2,), 7.0, dtype=torch.float64, device="cuda")
    args = lambda n: (ctypes.c_void_p(buf.data_ptr()), ctypes.c_void_p(buf.data_ptr()), ctypes.c_longlong(n),
                      ctypes.c_void_p(out.data_ptr()), None)
    for n in (nmax + 1, -1):
        assert lib.ov_blas_dot_static(*args(n)) == ovp.binding.OV_EINVAL
    assert lib.ov_blas_dot_static(*args(nmax + 1)) == ovp.binding.OV_EINVAL
    msg = lib.ov_blas_dot_static_error().decode()
    assert str(nmax) in msg and "exceeds" in msg
    assert lib.ov_blas_dot_static(None, None, ctypes.c_longlong(4), None, None) == ovp.binding.OV_EINVAL
    torch.cuda.synchronize()
    assert out.cpu().tolist() == [7.0, 7.0]
    assert lib.ov_blas_dot_static(*args(4)) == ovp.binding.OV_OK    # and a size that fits still works: <1,1> over 4
    torch.cuda.synchronize()
    assert out.cpu().tolist() == [4.0, 0.0]
