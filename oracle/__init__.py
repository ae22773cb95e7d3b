"""oracle -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

ctypes wrapper around ``oracle/clover_oracle.c`` (plain fp64 C, the CPU statement of what the
hot path of arXiv:1405.4524 computes; see the header of that file for citations and layouts).
Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It imports nothing from
``paper_1405_4524_b200`` and the CUDA path imports nothing from here.

Everything is numpy in / numpy out, canonical layouts:
  links   complex128 [4, T, Z, Y, X, 3, 3]
  spinor  complex128 [T, Z, Y, X, 4, 3]         (a batch adds a leading axis)
  clover  complex128 [T, Z, Y, X, 12, 12]
"""
import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "clover_oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")
_lib = None


def build(force=False):
    """Compile the oracle with gcc (OpenMP over sites only)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-std=c11", "-shared", "-fPIC", _SRC, "-o", _LIB, "-lm"])
    return _LIB


def lib():
    global _lib
    if _lib is None:
        build()
        _lib = ctypes.CDLL(_LIB)
        _lib.oracle_splitmix64.restype = ctypes.c_uint64
        _lib.oracle_splitmix64.argtypes = [ctypes.c_uint64, ctypes.c_uint64]
    return _lib


def _p(a):
    return a.ctypes.data_as(ctypes.c_void_p)


def _i4(v):
    return (ctypes.c_int * 4)(*[int(k) for k in v])


def _dims_of_links(U):
    _, T, Z, Y, X = U.shape[:5]
    return (X, Y, Z, T)


def _c(a):
    a = np.ascontiguousarray(a, dtype=np.complex128)
    return a


def threads():
    """Number of OpenMP threads the oracle will use."""
    return int(os.environ.get("OMP_NUM_THREADS", os.cpu_count() or 1))


def set_threads(n):
    """Set the OpenMP thread count of later oracle calls (bench.py reports a one-thread D-apply rate beside the all-cores one)."""
    lib()
    ctypes.CDLL("libgomp.so.1").omp_set_num_threads(int(n))
    os.environ["OMP_NUM_THREADS"] = str(int(n))


def hop(U, bc, psi):
    """(H psi)(x), SURVEY 8(c) O2."""
    U, psi = _c(U), _c(psi)
    out = np.empty_like(psi)
    lib().oracle_hop(_p(U), _i4(_dims_of_links(U)), _i4(bc), _p(psi), _p(out))
    return out


def fhat(U):
    """Fhat_{mu nu}(x) for the six planes 01 02 03 12 13 23: [6, T, Z, Y, X, 3, 3]."""
    U = _c(U)
    X, Y, Z, T = _dims_of_links(U)
    out = np.empty((6, T, Z, Y, X, 3, 3), dtype=np.complex128)
    lib().oracle_fhat(_p(U), _i4((X, Y, Z, T)), _p(out))
    return out


def clover_matrix(U, kappa, csw):
    """A(x) = 1 + i c_sw kappa sum_{mu<nu} sigma_{mu nu} (x) Fhat_{mu nu}: [T, Z, Y, X, 12, 12]."""
    U = _c(U)
    X, Y, Z, T = _dims_of_links(U)
    out = np.empty((T, Z, Y, X, 12, 12), dtype=np.complex128)
    lib().oracle_clover_matrix(_p(U), _i4((X, Y, Z, T)), ctypes.c_double(kappa), ctypes.c_double(csw), _p(out))
    return out


def clover_inverse(A):
    A = _c(A)
    out = np.empty_like(A)
    V = A.size // 144
    bad = lib().oracle_clover_inverse(_p(A), ctypes.c_long(V), _p(out))
    if bad:
        raise ArithmeticError(f"{bad} singular clover blocks")
    return out


def site_matvec(M, psi):
    """out(x) = M(x) psi(x) for a field of 12x12 matrices."""
    M, psi = _c(M), _c(psi)
    out = np.empty_like(psi)
    lib().oracle_site_matvec(_p(M), ctypes.c_long(M.size // 144), _p(psi), _p(out))
    return out


def apply_D(U, A, bc, kappa, psi):
    """D psi = A psi - kappa H psi, SURVEY 8(c) O4."""
    U, A, psi = _c(U), _c(A), _c(psi)
    out = np.empty_like(psi)
    lib().oracle_D(_p(U), _p(A), _i4(_dims_of_links(U)), _i4(bc), ctypes.c_double(kappa), _p(psi), _p(out))
    return out


def dense_D(U, A, bc, kappa):
    U, A = _c(U), _c(A)
    X, Y, Z, T = _dims_of_links(U)
    n = 12 * X * Y * Z * T
    M = np.empty((n, n), dtype=np.complex128)
    lib().oracle_dense_D(_p(U), _p(A), _i4((X, Y, Z, T)), _i4(bc), ctypes.c_double(kappa), _p(M))
    return M


def dense_inverse(M):
    M = _c(M)
    n = M.shape[0]
    out = np.empty_like(M)
    if lib().oracle_dense_inverse(_p(M), ctypes.c_int(n), _p(out)):
        raise ArithmeticError("singular matrix")
    return out


def bicgstab(U, A, bc, kappa, eta, tol=1e-12, max_iter=10000):
    """Textbook BiCGStab on the full, unpreconditioned system.

    Returns (psi, info) with info = dict(status, iters, true_resid)."""
    U, A, eta = _c(U), _c(A), _c(eta)
    psi = np.empty_like(eta)
    iters = ctypes.c_int(0)
    resid = ctypes.c_double(0.0)
    st = lib().oracle_bicgstab(_p(U), _p(A), _i4(_dims_of_links(U)), _i4(bc), ctypes.c_double(kappa), _p(eta),
                               _p(psi), ctypes.c_double(tol), ctypes.c_int(max_iter), ctypes.byref(iters),
                               ctypes.byref(resid))
    return psi, {"status": int(st), "iters": iters.value, "true_resid": resid.value}


def splitmix64(seed, ctr):
    return int(lib().oracle_splitmix64(ctypes.c_uint64(seed), ctypes.c_uint64(ctr)))


def noise_fill(dims, seed, n_rhs, rhs_offset=0, time_dilution=0, scale=1.0, dtype=np.float64, dilution=None):
    """Z4 sources, SURVEY 8(c) O5 / docs/NOISE.md: complex [n_rhs, T, Z, Y, X, 4, 3]."""
    X, Y, Z, T = dims
    if dilution is not None:      # bit 0 = time, bit 1 = spin-colour (docs/NOISE.md); time_dilution=1 is dilution=1
        time_dilution = dilution
    if dtype == np.float64:
        out = np.empty((n_rhs, T, Z, Y, X, 4, 3), dtype=np.complex128)
        lib().oracle_noise_fill(_p(out), _i4(dims), ctypes.c_uint64(seed), ctypes.c_int(n_rhs),
                                ctypes.c_int(rhs_offset), ctypes.c_int(time_dilution), ctypes.c_double(scale))
    else:
        out = np.empty((n_rhs, T, Z, Y, X, 4, 3), dtype=np.complex64)
        lib().oracle_noise_fill_f32(_p(out), _i4(dims), ctypes.c_uint64(seed), ctypes.c_int(n_rhs),
                                    ctypes.c_int(rhs_offset), ctypes.c_int(time_dilution), ctypes.c_float(scale))
    return out
