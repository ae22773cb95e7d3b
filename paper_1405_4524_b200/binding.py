"""Thin ctypes binding over the C-ABI of include/clover.h: argument marshalling only.

Every step of the path runs in the CUDA library ``libclover_b200.so`` (built in-tree by
``paper_1405_4524_b200.build``).  PyTorch is used for device memory and streams only.  Importing
this module fails loudly when the library is missing; there is no CPU fallback.
"""
import ctypes
import os

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libclover_b200.so")
if not os.path.exists(LIB_PATH):
    raise ImportError(f"{LIB_PATH} is missing: run `python -m paper_1405_4524_b200.build` (needs nvcc); there is no CPU fallback")
_lib = ctypes.CDLL(LIB_PATH)

OP_HOP_EO, OP_HOP_OE, OP_HOP_FULL, OP_CLOVER, OP_CLOVER_INV, OP_D_FULL, OP_MHAT = range(7)
KERNEL_HOP, KERNEL_AINV_HOP, KERNEL_A_MINUS_HOP, KERNEL_A_MINUS_HOP_S, KERNEL_A_MINUS_HOP_XW = range(5)
EXPORTS = ["clover_create", "clover_destroy", "dslash_apply", "clover_solve", "clover_solve_host", "noise_fill",
           "clover_bench_kernel", "clover_get_stats", "clover_last_error", "stochastic_operators", "stochastic_operators_noalloc", "stochastic_correlator", "stochastic_fill", "timeslice_norm2", "timeslice_inner"]


class ClovOpts(ctypes.Structure):
    _fields_ = [("recon", ctypes.c_int), ("max_rhs", ctypes.c_int)]


class RhsInfo(ctypes.Structure):
    _fields_ = [("status", ctypes.c_int), ("iters", ctypes.c_int), ("reliable_updates", ctypes.c_int),
                ("iter_resid", ctypes.c_double), ("true_resid", ctypes.c_double)]


class SolveStats(ctypes.Structure):
    _fields_ = [("kernel_launches", ctypes.c_longlong), ("ms_total", ctypes.c_double), ("ms_reorder", ctypes.c_double),
                ("ms_prep", ctypes.c_double), ("ms_iterate", ctypes.c_double), ("ms_reliable", ctypes.c_double),
                ("ms_finish", ctypes.c_double), ("n_ainv_hop", ctypes.c_longlong), ("n_a_minus_hop", ctypes.c_longlong),
                ("ms_ainv_hop", ctypes.c_double), ("ms_a_minus_hop", ctypes.c_double), ("n_a_minus_hop_s", ctypes.c_longlong),
                ("ms_a_minus_hop_s", ctypes.c_double), ("n_xrp_update", ctypes.c_longlong), ("ms_xrp_update", ctypes.c_double)]


_vp, _ip, _i, _d = ctypes.c_void_p, ctypes.POINTER(ctypes.c_int), ctypes.c_int, ctypes.c_double
_lib.clover_create.argtypes = [ctypes.POINTER(_vp), _vp, _ip, _d, _d, _ip, ctypes.POINTER(ClovOpts), _vp]
_lib.clover_destroy.argtypes = [_vp]
_lib.clover_destroy.restype = None
_lib.dslash_apply.argtypes = [_vp, _i, _i, _vp, _vp, _i, _vp]
_lib.clover_solve.argtypes = [_vp, _vp, _vp, _i, _d, _i, _i, _i, ctypes.POINTER(RhsInfo), _vp]
_lib.clover_solve_host.argtypes = [_vp, _vp, _vp, _i, _d, _i, _i, _i, ctypes.POINTER(RhsInfo), _vp]
_lib.noise_fill.argtypes = [_vp, _i, _ip, ctypes.c_uint64, _i, _i, _i, _d, _vp]
_lib.clover_bench_kernel.argtypes = [_vp, _i, _i, _i, _i, _i, ctypes.POINTER(ctypes.c_float), _vp]
_lib.clover_get_stats.argtypes = [_vp, ctypes.POINTER(SolveStats)]
_lib.clover_last_error.argtypes = [_vp]
_lib.stochastic_operators.argtypes = [_vp, _vp, _ip, _i, _vp, _vp]
_lib.stochastic_operators_noalloc.argtypes = [_vp, _vp, _ip, _i, _vp, _vp]
_lib.stochastic_correlator.argtypes = [_vp, _i, _i, _d, _vp, _vp]
_lib.stochastic_fill.argtypes = [_vp, _vp, _ip, _i, _i, _d, _i, _vp, _vp]
_lib.timeslice_norm2.argtypes = [_vp, ctypes.c_longlong, _i, ctypes.c_longlong, _vp, _vp]
_lib.timeslice_inner.argtypes = [_vp, _vp, ctypes.c_longlong, _i, ctypes.c_longlong, _vp, _vp]
_lib.clover_last_error.restype = ctypes.c_char_p


class CloverError(RuntimeError):
    pass


def _i4(v):
    return (ctypes.c_int * 4)(*[int(k) for k in v])


def _stream():
    return ctypes.c_void_p(torch.cuda.current_stream().cuda_stream)


def _check(rc):
    if rc < 0:
        raise CloverError(f"clover error {rc}: {_lib.clover_last_error(None).decode()}")
    return rc


def _require_cuda():
    if not torch.cuda.is_available():
        raise CloverError("no CUDA device: this library has no CPU fallback")


def _spinor_shape(dims, n_rhs):
    X, Y, Z, T = dims
    return (n_rhs, T, Z, Y, X, 4, 3)


def noise_fill(dims, seed, n_rhs, rhs_offset=0, time_dilution=0, scale=1.0, dtype=torch.complex128, out=None, dilution=None):
    """Z4 noise sources on the device: complex [n_rhs, T, Z, Y, X, 4, 3] (include/clover.h: noise_fill)."""
    _require_cuda()
    if dilution is not None:      # bit 0 = time, bit 1 = spin-colour; time_dilution=1 is dilution=1
        time_dilution = dilution
    if out is None:
        out = torch.empty(_spinor_shape(dims, n_rhs), dtype=dtype, device="cuda")
    assert out.is_cuda and out.is_contiguous() and out.dtype in (torch.complex64, torch.complex128)
    prec = 64 if out.dtype == torch.complex128 else 32
    _check(_lib.noise_fill(out.data_ptr(), prec, _i4(dims), seed, n_rhs, rhs_offset, int(time_dilution), float(scale), _stream()))
    return out


def stochastic_operators(eta, x):
    """O[t, i, j] = sum_y eta_i^*(t, y) gamma5 X_j(t, y) (paper eq. 7.6); eta, x complex128 [n, T, Z, Y, X, 4, 3] on the device."""
    _require_cuda()
    assert eta.is_cuda and x.is_cuda and eta.is_contiguous() and x.is_contiguous() and eta.dtype == x.dtype == torch.complex128
    assert eta.shape == x.shape
    n, T, Z, Y, X = eta.shape[:5]
    o = torch.empty((T, n, n), dtype=torch.complex128, device="cuda")
    _check(_lib.stochastic_operators(eta.data_ptr(), x.data_ptr(), _i4((X, Y, Z, T)), n, o.data_ptr(), _stream()))
    return o


NOALLOC_MAX_TNN = 1048576   # include/clover.h: CLOVER_NOALLOC_MAX_TNN


def stochastic_operators_noalloc(eta, x, out):
    """stochastic_operators without any allocation in the library (fixed internal scratch; T * n^2 <= NOALLOC_MAX_TNN): the caller
    passes the output `out` complex128 [T, n, n] on the device.  Calls that overlap on the GPU race on the shared scratch."""
    _require_cuda()
    assert eta.is_cuda and x.is_cuda and eta.is_contiguous() and x.is_contiguous() and eta.dtype == x.dtype == torch.complex128
    assert eta.shape == x.shape
    n, T, Z, Y, X = eta.shape[:5]
    assert out.is_cuda and out.is_contiguous() and out.dtype == torch.complex128 and tuple(out.shape) == (T, n, n)
    _check(_lib.stochastic_operators_noalloc(eta.data_ptr(), x.data_ptr(), _i4((X, Y, Z, T)), n, out.data_ptr(), _stream()))
    return out


def stochastic_correlator(o, scale=1.0):
    """C[t0, t] = (1 / (n^2 scale^4)) sum_ij O[t, i, j] O[t0, j, i] (paper eq. 7.7)."""
    _require_cuda()
    assert o.is_cuda and o.is_contiguous() and o.dtype == torch.complex128 and o.shape[1] == o.shape[2]
    T, n = o.shape[0], o.shape[1]
    c = torch.empty((T, T), dtype=torch.complex128, device="cuda")
    _check(_lib.stochastic_correlator(o.data_ptr(), T, n, float(scale), c.data_ptr(), _stream()))
    return c


def stochastic_fill(x, eta, t0=0, scale=1.0, dagger=False, out=None):
    """S[t, z3, a, x3, b] = (1/(n scale^2)) sum_i X_i(t, z3, a) conj(eta_i(t0, x3, b)) (paper eq. 7.3); dagger=True returns the
    Hermitian conjugate [x3, b, t, z3, a].  x, eta complex128 [n, T, Z, Y, X, 4, 3] on the device."""
    _require_cuda()
    assert x.is_cuda and eta.is_cuda and x.is_contiguous() and eta.is_contiguous() and x.dtype == eta.dtype == torch.complex128
    assert x.shape == eta.shape
    n, T, Z, Y, X = x.shape[:5]
    V3 = Z * Y * X
    shape = (V3, 12, T, V3, 12) if dagger else (T, V3, 12, V3, 12)
    if out is None:
        out = torch.empty(shape, dtype=torch.complex128, device="cuda")
    assert tuple(out.shape) == shape and out.is_contiguous()
    _check(_lib.stochastic_fill(x.data_ptr(), eta.data_ptr(), _i4((X, Y, Z, T)), n, int(t0), float(scale), int(dagger), out.data_ptr(), _stream()))
    return out


def timeslice_norm2(f, n_outer, T):
    """out[t] = sum |f[o, t, :]|^2 for a complex128 device tensor viewed as [n_outer, T, -1] (Table I traces)."""
    _require_cuda()
    assert f.is_cuda and f.is_contiguous() and f.dtype == torch.complex128 and f.numel() % (n_outer * T) == 0
    out = torch.empty(T, dtype=torch.float64, device="cuda")
    _check(_lib.timeslice_norm2(f.data_ptr(), n_outer, T, f.numel() // (n_outer * T), out.data_ptr(), _stream()))
    return out


def timeslice_inner(a, b, n_outer, T):
    """out[t] = sum a[o, t, :] conj(b[o, t, :]) for two complex128 device tensors viewed as [n_outer, T, -1]: the trace between
    fills from two independent source sets."""
    _require_cuda()
    assert a.is_cuda and a.is_contiguous() and a.dtype == torch.complex128 and a.numel() % (n_outer * T) == 0
    assert b.is_cuda and b.is_contiguous() and b.dtype == torch.complex128 and b.numel() == a.numel()
    out = torch.empty(T, dtype=torch.complex128, device="cuda")
    _check(_lib.timeslice_inner(a.data_ptr(), b.data_ptr(), n_outer, T, a.numel() // (n_outer * T), out.data_ptr(), _stream()))
    return out


class Clover:
    """A Wilson-clover operator context (include/clover.h: clover_create / clover_destroy)."""

    def __init__(self, gauge, kappa, csw, bc=(1, 1, 1, -1), recon=18, max_rhs=8):
        _require_cuda()
        assert gauge.is_cuda and gauge.dtype == torch.complex128 and gauge.is_contiguous() and gauge.shape[0] == 4
        _, T, Z, Y, X = gauge.shape[:5]
        self.dims = (X, Y, Z, T)
        self.kappa, self.csw, self.bc, self.recon, self.max_rhs = kappa, csw, tuple(bc), recon, max_rhs
        self._ctx = ctypes.c_void_p()
        opts = ClovOpts(recon, max_rhs)
        _check(_lib.clover_create(ctypes.byref(self._ctx), gauge.data_ptr(), _i4(self.dims), kappa, csw, _i4(bc), ctypes.byref(opts), _stream()))

    def close(self):
        if getattr(self, "_ctx", None) and _lib is not None:   # _lib is None during interpreter shutdown
            _lib.clover_destroy(self._ctx)
        self._ctx = None

    __del__ = close

    def dslash_apply(self, op, psi):
        """out = op(psi); psi complex64/128 [n_rhs, T, Z, Y, X, 4, 3] on the device."""
        assert psi.is_cuda and psi.is_contiguous() and psi.dtype in (torch.complex64, torch.complex128)
        assert tuple(psi.shape[1:]) == _spinor_shape(self.dims, 1)[1:]
        out = torch.empty_like(psi)
        prec = 64 if psi.dtype == torch.complex128 else 32
        _check(_lib.dslash_apply(self._ctx, op, prec, psi.data_ptr(), out.data_ptr(), psi.shape[0], _stream()))
        return out

    def _solve(self, fn, sources, out, tol, max_iter, batch, mixed):
        n = sources.shape[0]
        info = (RhsInfo * max(n, 1))()
        bad = _check(fn(self._ctx, sources.data_ptr(), out.data_ptr(), n, tol, max_iter, batch, int(mixed), info, _stream()))
        infos = [dict(status=i.status, iters=i.iters, reliable_updates=i.reliable_updates, iter_resid=i.iter_resid, true_resid=i.true_resid)
                 for i in info[:n]]
        return out, infos, bad

    def solve(self, sources, tol=1e-10, max_iter=1000, batch=None, mixed=True, out=None):
        """D psi_r = eta_r for device sources complex128 [n_rhs, T, Z, Y, X, 4, 3] -> (psi, infos, n_bad)."""
        assert sources.is_cuda and sources.is_contiguous() and sources.dtype == torch.complex128
        if out is None:
            out = torch.empty_like(sources)
        return self._solve(_lib.clover_solve, sources, out, tol, max_iter, batch or self.max_rhs, mixed)

    def solve_host(self, sources, tol=1e-10, max_iter=1000, batch=None, mixed=True, out=None):
        """Same from HOST tensors (pinned for speed); copies run inside the call."""
        assert (not sources.is_cuda) and sources.is_contiguous() and sources.dtype == torch.complex128
        if out is None:
            out = torch.empty_like(sources, pin_memory=True)
        return self._solve(_lib.clover_solve_host, sources, out, tol, max_iter, batch or self.max_rhs, mixed)

    def bench_kernel(self, kernel, precision, n_rhs, reps=20, flush_l2=False):
        ms = ctypes.c_float(0)
        _check(_lib.clover_bench_kernel(self._ctx, kernel, precision, n_rhs, reps, int(flush_l2), ctypes.byref(ms), _stream()))
        return ms.value

    def stats(self):
        s = SolveStats()
        _check(_lib.clover_get_stats(self._ctx, ctypes.byref(s)))
        return {k: getattr(s, k) for k, _ in SolveStats._fields_}
