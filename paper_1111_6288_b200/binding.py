"""Thin ctypes binding of libov.so (include/ov.h): argument marshalling only.

Every step of the path runs in the CUDA kernels behind the C ABI; torch is used here for device memory
and streams.  There is no CPU fallback: if libov.so is missing or no CUDA device is usable, calls raise.
Method names mirror the C entry points (ov_apply_hw -> Overlap.apply_hw, ...).
"""
from __future__ import annotations

import ctypes
import os

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libov.so")

OV_OK, OV_EINVAL, OV_ENOMEM, OV_ECUDA, OV_ESTATE, OV_ENOCONV = range(6)
_CODES = {1: "OV_EINVAL", 2: "OV_ENOMEM", 3: "OV_ECUDA", 4: "OV_ESTATE", 5: "OV_ENOCONV"}

# every symbol include/ov.h declares (tests check that the library exports all of them)
SYMBOLS = [
    "ov_create", "ov_create_ex", "ov_destroy", "ov_last_error", "ov_spinor_bytes", "ov_volume", "ov_spinor_layout", "ov_launch_count",
    "ov_timing_enable", "ov_timing_read",
    "ov_set_dslash_variant", "ov_get_dslash_variant", "ov_pack_spinor", "ov_unpack_spinor", "ov_dslash", "ov_apply_hw",
    "ov_chebyshev_coeffs", "ov_set_polynomial", "ov_set_smallspace", "ov_project", "ov_apply_sign",
    "ov_apply_dov", "ov_apply_dov_reduced", "ov_apply_hw_f32", "ov_set_cg_adaptive", "ov_cg_orders", "ov_apply_hw_host", "ov_apply_dov_host", "ov_blas_axpy", "ov_blas_scale", "ov_blas_dot",
    "ov_blas_norm2", "ov_multishift_cg", "ov_lanczos_lowmodes", "ov_lanczos_stats", "ov_lanczos_dov_lowmodes", "ov_set_deflation", "ov_set_cg_operator", "ov_cg_chirality", "ov_host_eigh",
    "ov_blas_dot_static", "ov_blas_dot_static_max", "ov_blas_dot_static_error",
]


class OvError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"{_CODES.get(code, code)}: {msg}")
        self.code = code


_lib = None


def load_library():
    """Loads libov.so; raises (never falls back) if it has not been built."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise OvError(OV_ESTATE, f"{LIB_PATH} not built: run `python -m paper_1111_6288_b200.build`")
        lib = ctypes.CDLL(LIB_PATH)
        lib.ov_last_error.restype = ctypes.c_char_p
        lib.ov_spinor_bytes.restype = ctypes.c_size_t
        lib.ov_volume.restype = ctypes.c_longlong
        lib.ov_launch_count.restype = ctypes.c_longlong
        lib.ov_destroy.restype = None
        lib.ov_blas_dot_static_max.restype = ctypes.c_longlong
        lib.ov_blas_dot_static_error.restype = ctypes.c_char_p
        _lib = lib
    return _lib


def _ptr(t):
    if isinstance(t, torch.Tensor):
        assert t.is_contiguous(), "tensor must be contiguous"
        return ctypes.c_void_p(t.data_ptr())
    if isinstance(t, np.ndarray):
        assert t.flags["C_CONTIGUOUS"]
        return ctypes.c_void_p(t.ctypes.data)
    raise TypeError(type(t))


def _darr(a):
    a = np.ascontiguousarray(a, dtype=np.float64)
    return a, a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def chebyshev_coeffs(order: int, eps: float) -> np.ndarray:
    """ov_chebyshev_coeffs: Chebyshev-interpolation coefficients of x^(-1/2) on [eps,1] (host helper)."""
    out = np.empty(order + 1, dtype=np.float64)
    rc = load_library().ov_chebyshev_coeffs(ctypes.c_int(order), ctypes.c_double(eps),
                                            out.ctypes.data_as(ctypes.POINTER(ctypes.c_double)))
    if rc != OV_OK:
        raise OvError(rc, "ov_chebyshev_coeffs")
    return out


def host_eigh(A: np.ndarray):
    """ov_host_eigh: the library's host Jacobi eigensolver (test hook)."""
    A = np.ascontiguousarray(A, dtype=np.complex128)
    n = A.shape[0]
    w = np.empty(n)
    Z = np.empty((n, n), dtype=np.complex128)
    rc = load_library().ov_host_eigh(ctypes.c_int(n), _ptr(A), w.ctypes.data_as(ctypes.POINTER(ctypes.c_double)), _ptr(Z))
    if rc != OV_OK:
        raise OvError(rc, "ov_host_eigh")
    return w, Z


def blas_dot_static_max() -> int:
    """ov_blas_dot_static_max: the longest vector (complex elements) ov_blas_dot_static accepts."""
    return int(load_library().ov_blas_dot_static_max())


def blas_dot_static(x, y, out, stream=None):
    """ov_blas_dot_static: <x, y> = sum conj(x) y without any device allocation, for programs that cannot call cudaMalloc
    (all of HBM already in their own pool, or other streams that a cudaMalloc would stall); see include/ov.h.

    x, y: contiguous complex128 CUDA tensors of equal length (any shape); out: a CUDA tensor of 2 float64 (or 1
    complex128) that the CALLER provides -- this wrapper allocates nothing either -- and that receives (re, im) once
    `stream` (default: torch's current stream) gets there; nothing is synchronised.  Raises OvError(OV_EINVAL) for more
    than blas_dot_static_max() elements.  The scratch array behind it is shared per GPU: keep calls on one stream."""
    if not torch.cuda.is_available():
        raise OvError(OV_ECUDA, "no CUDA device: this library has no CPU fallback")
    lib = load_library()
    assert x.is_cuda and y.is_cuda and out.is_cuda and x.dtype == y.dtype == torch.complex128
    assert x.numel() == y.numel() and out.numel() * out.element_size() == 16
    stream = stream if stream is not None else torch.cuda.current_stream(x.device)
    with torch.cuda.device(x.device):
        rc = lib.ov_blas_dot_static(_ptr(x), _ptr(y), ctypes.c_longlong(x.numel()), _ptr(out),
                                    ctypes.c_void_p(stream.cuda_stream))
    if rc != OV_OK:
        raise OvError(rc, lib.ov_blas_dot_static_error().decode())
    return out


class OvOptions(ctypes.Structure):
    """struct ov_options of include/ov.h."""
    _fields_ = [("layout", ctypes.c_int), ("t_boundary", ctypes.c_int), ("wall_mask", ctypes.c_int),
                ("field", ctypes.c_int), ("field_origin", ctypes.c_int), ("reserved", ctypes.c_int),
                ("field_qE", ctypes.c_double)]


class Overlap:
    """One ov_ctx.  Spinor arguments are torch complex128 CUDA tensors in the ABI layout [nrhs?][12][V]
    unless a method says "canonical" ([T][Z][Y][X][4][3])."""

    LAYOUTS = {"auto": 0, "blocked": 1, "planes": 2}
    BOUNDARIES = {"antiperiodic": 0, "periodic": 1, "open": 2}

    def __init__(self, dims, kappa, gauge, recon=18, stream=None, layout="auto", t_boundary="antiperiodic",
                 walls=(), field_dir=None, field_qE=0.0, field_origin=0):
        """walls: space directions (0, 1, 2) with a Dirichlet wall; field_dir: direction of a constant electric
        field of strength field_qE (None = no field).  See ov_options in include/ov.h."""
        if not torch.cuda.is_available():
            raise OvError(OV_ECUDA, "no CUDA device: this library has no CPU fallback")
        self.lib = load_library()
        self.dims = tuple(int(d) for d in dims)
        self.V = int(np.prod(self.dims))
        if isinstance(gauge, np.ndarray):
            gauge = torch.from_numpy(np.ascontiguousarray(gauge, dtype=np.complex128)).cuda()
        assert gauge.dtype == torch.complex128 and gauge.is_cuda and gauge.numel() == self.V * 36
        self.device = gauge.device
        self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        self._ctx = ctypes.c_void_p()
        cdims = (ctypes.c_int * 4)(*self.dims)
        opt = OvOptions(self.LAYOUTS[layout], self.BOUNDARIES[t_boundary], sum(1 << int(mu) for mu in walls),
                        0 if field_dir is None else int(field_dir) + 1, int(field_origin), 0, float(field_qE))
        rc = self.lib.ov_create_ex(ctypes.byref(self._ctx), cdims, ctypes.c_double(kappa), _ptr(gauge.contiguous()),
                                   ctypes.c_int(recon), ctypes.c_void_p(self.stream.cuda_stream), ctypes.byref(opt))
        if rc != OV_OK:
            raise OvError(rc, "ov_create failed")
        self._keepalive = None

    def close(self):
        if getattr(self, "_ctx", None) is not None and self._ctx:
            self.lib.ov_destroy(self._ctx)
            self._ctx = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check(self, rc):
        if rc != OV_OK:
            raise OvError(rc, self.lib.ov_last_error(self._ctx).decode())

    # ---- helpers
    def new_spinor(self, nrhs=None):
        shape = (12, self.V) if nrhs is None else (nrhs, 12, self.V)
        return torch.empty(shape, dtype=torch.complex128, device=self.device)

    @staticmethod
    def _nrhs(t):
        return 1 if t.dim() == 2 else t.shape[0]

    @property
    def spinor_layout(self):
        """1 = blocked [V/32][12][32], 0 = planes [12][V] (include/ov.h, Layouts)."""
        return int(self.lib.ov_spinor_layout(self._ctx))

    @property
    def launch_count(self):
        return int(self.lib.ov_launch_count(self._ctx))

    def timing_enable(self, on=True):
        self._check(self.lib.ov_timing_enable(self._ctx, ctypes.c_int(1 if on else 0)))

    def timing_read(self):
        """{wilson_ms, wilson_launches, projector_ms, projector_launches} since the last read."""
        out = (ctypes.c_double * 4)()
        self._check(self.lib.ov_timing_read(self._ctx, out))
        return dict(wilson_ms=out[0], wilson_launches=int(out[1]), projector_ms=out[2], projector_launches=int(out[3]))

    @property
    def dslash_variant(self):
        return int(self.lib.ov_get_dslash_variant(self._ctx))

    def set_dslash_variant(self, v):
        self._check(self.lib.ov_set_dslash_variant(self._ctx, ctypes.c_int(v)))

    # ---- layout
    def pack_spinor(self, canonical):
        """canonical [nrhs?][T][Z][Y][X][4][3] (device) -> ABI"""
        c = canonical.contiguous()
        nrhs = c.numel() // (12 * self.V)
        out = self.new_spinor(None if c.dim() == 6 else nrhs)
        self._check(self.lib.ov_pack_spinor(self._ctx, _ptr(c), _ptr(out), ctypes.c_int(nrhs)))
        return out

    def unpack_spinor(self, abi):
        nrhs = self._nrhs(abi)
        X, Y, Z, T = self.dims
        shape = (T, Z, Y, X, 4, 3) if abi.dim() == 2 else (nrhs, T, Z, Y, X, 4, 3)
        out = torch.empty(shape, dtype=torch.complex128, device=self.device)
        self._check(self.lib.ov_unpack_spinor(self._ctx, _ptr(abi), _ptr(out), ctypes.c_int(nrhs)))
        return out

    # ---- operator
    def _apply(self, fn, x, out, *pre):
        out = torch.empty_like(x) if out is None else out
        self._check(fn(self._ctx, *pre, _ptr(x), _ptr(out), ctypes.c_int(self._nrhs(x))))
        return out

    def dslash(self, x, out=None):
        return self._apply(self.lib.ov_dslash, x, out)

    def apply_hw(self, x, out=None):
        return self._apply(self.lib.ov_apply_hw, x, out)

    def apply_sign(self, x, out=None):
        return self._apply(self.lib.ov_apply_sign, x, out)

    def apply_dov(self, mass, x, out=None):
        return self._apply(self.lib.ov_apply_dov, x, out, ctypes.c_double(mass))

    def apply_dov_reduced(self, mass, x, order, use_f32, out=None):
        out = torch.empty_like(x) if out is None else out
        self._check(self.lib.ov_apply_dov_reduced(self._ctx, ctypes.c_double(mass), _ptr(x), _ptr(out), ctypes.c_int(order),
                                                  ctypes.c_int(1 if use_f32 else 0)))
        return out

    def apply_hw_f32(self, x, out=None):
        out = torch.empty_like(x) if out is None else out
        self._check(self.lib.ov_apply_hw_f32(self._ctx, _ptr(x), _ptr(out)))
        return out

    def set_cg_adaptive(self, mode):
        self._check(self.lib.ov_set_cg_adaptive(self._ctx, ctypes.c_int(mode)))

    def cg_orders(self):
        buf = (ctypes.c_int * 4096)()
        n = self.lib.ov_cg_orders(self._ctx, buf, ctypes.c_int(4096))
        return [buf[i] for i in range(min(n, 4096))]

    def apply_hw_host(self, x_host, out_host=None):
        """canonical HOST array (numpy or torch, pinned for asynchronous copies) in, canonical HOST array out (H2D and
        D2H inside the call)."""
        x = x_host if isinstance(x_host, torch.Tensor) else np.ascontiguousarray(x_host, dtype=np.complex128)
        if out_host is None:
            out_host = torch.empty_like(x) if isinstance(x, torch.Tensor) else np.empty_like(x)
        nrhs = (x.numel() if isinstance(x, torch.Tensor) else x.size) // (12 * self.V)
        self._check(self.lib.ov_apply_hw_host(self._ctx, _ptr(x), _ptr(out_host), ctypes.c_int(nrhs)))
        return out_host

    def apply_dov_host(self, mass, x_host, out_host=None):
        x = x_host if isinstance(x_host, torch.Tensor) else np.ascontiguousarray(x_host, dtype=np.complex128)
        if out_host is None:
            out_host = torch.empty_like(x) if isinstance(x, torch.Tensor) else np.empty_like(x)
        nrhs = (x.numel() if isinstance(x, torch.Tensor) else x.size) // (12 * self.V)
        self._check(self.lib.ov_apply_dov_host(self._ctx, ctypes.c_double(mass), _ptr(x), _ptr(out_host),
                                               ctypes.c_int(nrhs)))
        return out_host

    def set_polynomial(self, coeffs, eps, norm):
        c, pc = _darr(coeffs)
        self._check(self.lib.ov_set_polynomial(self._ctx, pc, ctypes.c_int(len(c) - 1), ctypes.c_double(eps),
                                               ctypes.c_double(norm)))

    def set_smallspace(self, V, lam):
        """V: [k][12][V] ABI spinors on the device (borrowed: kept alive here), lam: k eigenvalues of Q."""
        if V is None or len(lam) == 0:
            self._check(self.lib.ov_set_smallspace(self._ctx, None, None, ctypes.c_int(0)))
            self._keepalive = None
            return
        l, pl = _darr(lam)
        assert V.is_contiguous() and V.shape[0] == len(l)
        self._check(self.lib.ov_set_smallspace(self._ctx, _ptr(V), pl, ctypes.c_int(len(l))))
        self._keepalive = V

    def project(self, x):
        perp, low = torch.empty_like(x), torch.empty_like(x)
        k = self._keepalive.shape[0]
        coef = np.empty(2 * k)
        self._check(self.lib.ov_project(self._ctx, _ptr(x), _ptr(perp), _ptr(low),
                                        coef.ctypes.data_as(ctypes.POINTER(ctypes.c_double))))
        return perp, low, coef.view(np.complex128)

    # ---- BLAS-1
    def blas_axpy(self, a, x, y):
        a = complex(a)
        self._check(self.lib.ov_blas_axpy(self._ctx, ctypes.c_double(a.real), ctypes.c_double(a.imag), _ptr(x), _ptr(y)))

    def blas_scale(self, a, x):
        self._check(self.lib.ov_blas_scale(self._ctx, ctypes.c_double(a), _ptr(x)))

    def blas_dot(self, x, y) -> complex:
        out = (ctypes.c_double * 2)()
        self._check(self.lib.ov_blas_dot(self._ctx, _ptr(x), _ptr(y), out))
        return complex(out[0], out[1])

    def blas_norm2(self, x) -> float:
        out = ctypes.c_double()
        self._check(self.lib.ov_blas_norm2(self._ctx, _ptr(x), ctypes.byref(out)))
        return out.value

    # ---- consumers
    def multishift_cg(self, masses, b, tol=1e-8, maxiter=1000, true_residuals=True):
        """x[nmass], iterations, true relative residuals (None if not asked for), converged"""
        m, pm = _darr(masses)
        x = self.new_spinor(len(m))
        iters = ctypes.c_int()
        res = np.empty(len(m)) if true_residuals else None
        pres = res.ctypes.data_as(ctypes.POINTER(ctypes.c_double)) if true_residuals else None
        rc = self.lib.ov_multishift_cg(self._ctx, pm, ctypes.c_int(len(m)), _ptr(b), _ptr(x), ctypes.c_double(tol),
                                       ctypes.c_int(maxiter), ctypes.byref(iters), pres)
        if rc not in (OV_OK, OV_ENOCONV):
            self._check(rc)
        return x, iters.value, res, rc == OV_OK

    def lanczos_lowmodes(self, k, tol=1e-8, max_restarts=50, cheb_order=100, subspace=0):
        V = self.new_spinor(k)
        lam, res = np.empty(k), np.empty(k)
        rc = self.lib.ov_lanczos_lowmodes(self._ctx, ctypes.c_int(k), ctypes.c_double(tol), ctypes.c_int(max_restarts),
                                          ctypes.c_int(cheb_order), ctypes.c_int(subspace), _ptr(V),
                                          lam.ctypes.data_as(ctypes.POINTER(ctypes.c_double)),
                                          res.ctypes.data_as(ctypes.POINTER(ctypes.c_double)))
        if rc not in (OV_OK, OV_ENOCONV):
            self._check(rc)
        return V, lam, res, rc == OV_OK

    def lanczos_dov_lowmodes(self, chirality, k, tol=1e-9, max_restarts=50, cheb_order=12, subspace=0):
        """ov_lanczos_dov_lowmodes: k lowest eigenpairs of D_ov^+ D_ov in one chirality sector (+1 / -1)."""
        W = self.new_spinor(k)
        mu, res = np.empty(k), np.empty(k)
        rc = self.lib.ov_lanczos_dov_lowmodes(self._ctx, ctypes.c_int(chirality), ctypes.c_int(k), ctypes.c_double(tol),
                                              ctypes.c_int(max_restarts), ctypes.c_int(cheb_order), ctypes.c_int(subspace),
                                              _ptr(W), mu.ctypes.data_as(ctypes.POINTER(ctypes.c_double)),
                                              res.ctypes.data_as(ctypes.POINTER(ctypes.c_double)))
        if rc not in (OV_OK, OV_ENOCONV):
            self._check(rc)
        return W, mu, res, rc == OV_OK

    def set_cg_operator(self, mode):
        """ov_set_cg_operator: 0 = gamma5 D gamma5 D, 1 = chirally symmetric form (one sign per step for a chiral source)."""
        self._check(self.lib.ov_set_cg_operator(self._ctx, ctypes.c_int(mode)))

    @property
    def cg_chirality(self):
        return int(self.lib.ov_cg_chirality(self._ctx))

    def set_deflation(self, W, mu):
        """ov_set_deflation: W [k][12][V] eigenvectors of D_ov^+ D_ov (kept alive here), mu their eigenvalues; None clears."""
        if W is None:
            self._check(self.lib.ov_set_deflation(self._ctx, None, None, ctypes.c_int(0)))
            self._defl = None
            return
        mu = np.ascontiguousarray(mu, dtype=np.float64)
        assert W.is_cuda and W.dtype == torch.complex128 and W.is_contiguous() and W.shape[0] == len(mu)
        self._check(self.lib.ov_set_deflation(self._ctx, _ptr(W), mu.ctypes.data_as(ctypes.POINTER(ctypes.c_double)),
                                              ctypes.c_int(len(mu))))
        self._defl = W

    def lanczos_stats(self):
        """ov_lanczos_stats: counters of the last lanczos_lowmodes call."""
        out = (ctypes.c_double * 12)()
        self._check(self.lib.ov_lanczos_stats(self._ctx, out))
        return dict(restarts=int(out[0]), filter_applies=int(out[1]), launches=int(out[2]), edge=out[3],
                    widenings=int(out[4]), subspace=int(out[5]),
                    seconds=dict(host_eigh=out[6], filter=out[7], orthogonalisation=out[8], rotation=out[9],
                                 rayleigh_ritz=out[10], total=out[11]))
