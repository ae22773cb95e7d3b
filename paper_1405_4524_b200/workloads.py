"""Seeded synthetic inputs shared by the tests, bench.py and smoke().

This module holds NONE of the method's arithmetic: only the BASELINE.json workload table and
the gauge-link generator U = exp(i eps H).  It is the one module both the oracle-side and the
CUDA-side callers may import (numpy only).  The links stand in for the paper's quenched
beta = 5.96 ensemble, which is not available; recipe = DESIGN.md "Inputs".
"""
import numpy as np

# BASELINE.json configs[0..4]; bc = periodic space, antiperiodic time; scale = 1/sqrt2 literal.
INV_SQRT2 = float.fromhex("0x1.6a09e667f3bcdp-1")  # 0x3FE6A09E667F3BCD
CONFIGS = [
    dict(name="cfg0_4x4x4x8", dims=(4, 4, 4, 8), eps=0.2, kappa=0.120, csw=1.0, n_rhs=1, batch=1, mixed=0,
         recon=18, dilution=0, gauge_seed=1000, noise_seed=2000),
    dict(name="cfg1_8x8x8x16", dims=(8, 8, 8, 16), eps=0.3, kappa=0.120, csw=1.0, n_rhs=4, batch=4, mixed=0,
         recon=18, dilution=0, gauge_seed=1001, noise_seed=2001),
    dict(name="cfg2_16x16x16x32", dims=(16, 16, 16, 32), eps=0.4, kappa=0.118, csw=1.5, n_rhs=16, batch=4, mixed=1,
         recon=18, dilution=0, gauge_seed=1002, noise_seed=2002),
    dict(name="cfg3_24x24x24x48", dims=(24, 24, 24, 48), eps=0.4, kappa=0.118, csw=1.5, n_rhs=32, batch=8, mixed=1,
         recon=18, dilution=0, gauge_seed=1003, noise_seed=2003),
    dict(name="cfg4_32x32x32x64", dims=(32, 32, 32, 64), eps=0.5, kappa=0.115, csw=1.8, n_rhs=64, batch=8, mixed=1,
         recon=12, dilution=1, gauge_seed=1004, noise_seed=2004),
]
BC = (1, 1, 1, -1)
TOL = 1e-10

# Gell-Mann matrices lambda_1..lambda_8
_GM = np.zeros((8, 3, 3), dtype=np.complex128)
_GM[0][0, 1] = _GM[0][1, 0] = 1
_GM[1][0, 1] = -1j
_GM[1][1, 0] = 1j
_GM[2][0, 0] = 1
_GM[2][1, 1] = -1
_GM[3][0, 2] = _GM[3][2, 0] = 1
_GM[4][0, 2] = -1j
_GM[4][2, 0] = 1j
_GM[5][1, 2] = _GM[5][2, 1] = 1
_GM[6][1, 2] = -1j
_GM[6][2, 1] = 1j
_GM[7][0, 0] = _GM[7][1, 1] = 1 / np.sqrt(3)
_GM[7][2, 2] = -2 / np.sqrt(3)


def random_su3_algebra(rng, n):
    """n traceless Hermitian 3x3 matrices H = sum_a h_a lambda_a / 2, h_a ~ N(0,1) iid."""
    h = rng.standard_normal((n, 8))
    return np.einsum("na,aij->nij", h, _GM) / 2


def expi(H, eps):
    """exp(i eps H) for a batch of Hermitian matrices, via the Hermitian eigendecomposition
    (exactly unitary; det = 1 when tr H = 0)."""
    w, v = np.linalg.eigh(H)
    return np.einsum("nij,nj,nkj->nik", v, np.exp(1j * eps * w), v.conj())


def gauge_links(dims, eps, seed, chunk=1 << 18):
    """U_mu(x) = exp(i eps H_mu(x)), canonical layout complex128 [4, T, Z, Y, X, 3, 3]."""
    X, Y, Z, T = dims
    n = 4 * T * Z * Y * X
    rng = np.random.default_rng(seed)
    U = np.empty((n, 3, 3), dtype=np.complex128)
    for a in range(0, n, chunk):
        b = min(n, a + chunk)
        U[a:b] = expi(random_su3_algebra(rng, b - a), eps)
    return U.reshape(4, T, Z, Y, X, 3, 3)


def unit_links(dims):
    X, Y, Z, T = dims
    U = np.zeros((4, T, Z, Y, X, 3, 3), dtype=np.complex128)
    U[..., 0, 0] = U[..., 1, 1] = U[..., 2, 2] = 1
    return U


def random_su3_field(dims, seed):
    """One random SU(3) matrix per site (a gauge transformation g(x)): [T, Z, Y, X, 3, 3]."""
    X, Y, Z, T = dims
    rng = np.random.default_rng(seed)
    return expi(random_su3_algebra(rng, T * Z * Y * X), 1.0).reshape(T, Z, Y, X, 3, 3)


def random_spinor(dims, seed, n_rhs=None):
    """Gaussian complex spinor field(s): [T, Z, Y, X, 4, 3] or [n_rhs, ...]."""
    X, Y, Z, T = dims
    rng = np.random.default_rng(seed)
    shape = (T, Z, Y, X, 4, 3) if n_rhs is None else (n_rhs, T, Z, Y, X, 4, 3)
    return rng.standard_normal(shape) + 1j * rng.standard_normal(shape)


def parity_mask(dims):
    """(x+y+z+t) mod 2 as an int array [T, Z, Y, X]; even sites = 0."""
    X, Y, Z, T = dims
    t, z, y, x = np.meshgrid(np.arange(T), np.arange(Z), np.arange(Y), np.arange(X), indexing="ij")
    return (t + z + y + x) & 1
