"""Pins for the CPU oracle (CPU only).  Each test checks oracle/ against something the paper or
the mathematics fix -- never against itself and never against the CUDA path.

P1 free-field closed form      (BASELINE.json north_star check 1)
P2 gamma5-hermiticity          (check 2; PAPER.md L293 uses it)
P3 gauge covariance            (check 3)
P4 2^4 dense inverse/estimator (check 4; eq. 7.3 "1/sqrt(N_r)")   -> test_oracle_dense.py
P5 abelian closed form of Fhat (leaf geometry, orientation, the 1/8)
P6 tree-level O(a) improvement (sign and size of the clover term; "tree-level improved ... c_SW = 1.0")
P7 structure of A              (Hermitian, commutes with gamma5, chirality blocks)
"""
import numpy as np
import pytest

import oracle
from gammas import GAMMA, GAMMA5, sigma
from paper_1405_4524_b200 import workloads as wl


def _momenta(dims, bc, n):
    return np.array([2 * np.pi * (n[m] + (0.5 if bc[m] < 0 else 0.0)) / dims[m] for m in range(4)])


def _plane_wave(dims, p):
    X, Y, Z, T = dims
    t, z, y, x = np.meshgrid(np.arange(T), np.arange(Z), np.arange(Y), np.arange(X), indexing="ij")
    return np.exp(1j * (p[0] * x + p[1] * y + p[2] * z + p[3] * t))


def _D_of_p(p, kappa):
    a = 1 - 2 * kappa * np.sum(np.cos(p))
    return a * np.eye(4) + 2j * kappa * sum(GAMMA[m] * np.sin(p[m]) for m in range(4))


def _S_of_p(p, kappa):
    a = 1 - 2 * kappa * np.sum(np.cos(p))
    num = a * np.eye(4) - 2j * kappa * sum(GAMMA[m] * np.sin(p[m]) for m in range(4))
    return num / (a * a + 4 * kappa ** 2 * np.sum(np.sin(p) ** 2))


@pytest.mark.parametrize("bc", [(1, 1, 1, -1), (1, 1, 1, 1), (-1, 1, -1, 1)])
def test_P1_free_field_plane_wave(bc):
    """Unit links: A = 1 for any c_sw, and D e^{ipx} u = e^{ipx} D(p) u."""
    dims, kappa = (4, 6, 4, 8), 0.12
    U = wl.unit_links(dims)
    A = oracle.clover_matrix(U, kappa, 1.7)
    assert np.abs(A - np.eye(12)).max() == 0.0
    rng = np.random.default_rng(5)
    for n in [(1, 2, 3, 5), (0, 0, 0, 0), (3, 5, 1, 7)]:
        p = _momenta(dims, bc, n)
        u = rng.standard_normal(4) + 1j * rng.standard_normal(4)
        w = rng.standard_normal(3) + 1j * rng.standard_normal(3)
        pw = _plane_wave(dims, p)
        psi = pw[..., None, None] * u[:, None] * w[None, :]
        got = oracle.apply_D(U, A, bc, kappa, psi)
        want = pw[..., None, None] * (_D_of_p(p, kappa) @ u)[:, None] * w[None, :]
        assert np.abs(got - want).max() < 1e-13


def test_P1_free_field_point_propagator():
    """Point-source solve = (1/V) sum_p e^{ip.x} S(p), S(p) = [a - 2i kappa gamma.sin p]/[a^2 + 4 kappa^2 sin^2 p]."""
    dims, kappa, bc = (4, 4, 4, 8), 0.12, (1, 1, 1, -1)
    X, Y, Z, T = dims
    U = wl.unit_links(dims)
    A = oracle.clover_matrix(U, kappa, 1.0)
    s0, c0 = 2, 1
    eta = np.zeros((T, Z, Y, X, 4, 3), dtype=complex)
    eta[0, 0, 0, 0, s0, c0] = 1
    psi, info = oracle.bicgstab(U, A, bc, kappa, eta, tol=1e-13)
    assert info["status"] == 0 and info["true_resid"] < 1e-12
    want = np.zeros((T, Z, Y, X, 4), dtype=complex)
    for nx in range(X):
        for ny in range(Y):
            for nz in range(Z):
                for nt in range(T):
                    p = _momenta(dims, bc, (nx, ny, nz, nt))
                    want += _plane_wave(dims, p)[..., None] * _S_of_p(p, kappa)[:, s0]
    want /= X * Y * Z * T
    assert np.abs(psi[..., c0] - want).max() < 1e-11
    other = [c for c in range(3) if c != c0]
    assert np.abs(psi[..., other]).max() < 1e-12


def _setup(dims=(4, 4, 4, 8), eps=0.3, seed=11, kappa=0.12, csw=1.0):
    U = wl.gauge_links(dims, eps, seed)
    A = oracle.clover_matrix(U, kappa, csw)
    return U, A


def test_P2_gamma5_hermiticity():
    dims, kappa, bc = (4, 4, 4, 8), 0.12, (1, 1, 1, -1)
    U, A = _setup(dims, kappa=kappa)
    x = wl.random_spinor(dims, 1)
    y = wl.random_spinor(dims, 2)
    g5 = np.diag(GAMMA5).real[:, None]
    lhs = np.vdot(y, oracle.apply_D(U, A, bc, kappa, x))
    rhs = np.vdot(g5 * oracle.apply_D(U, A, bc, kappa, g5 * y), x)
    assert abs(lhs - rhs) / abs(lhs) < 1e-13
    # and for the hop alone (pairs the +mu and -mu terms)
    lhs = np.vdot(y, oracle.hop(U, bc, x))
    rhs = np.vdot(g5 * oracle.hop(U, bc, g5 * y), x)
    assert abs(lhs - rhs) / abs(lhs) < 1e-13


def _gauge_transform(U, g):
    """U'_mu(x) = g(x) U_mu(x) g(x+mu)^dagger; axes of the site array are (t,z,y,x)."""
    Up = np.empty_like(U)
    for mu in range(4):
        gp = np.roll(g, -1, axis=3 - mu)
        Up[mu] = np.einsum("...ab,...bc,...dc->...ad", g, U[mu], gp.conj())
    return Up


def test_P3_gauge_covariance():
    dims, kappa, csw = (4, 6, 4, 8), 0.118, 1.5
    for bc in [(1, 1, 1, -1), (1, 1, 1, 1)]:
        U = wl.gauge_links(dims, 0.4, 21)
        g = wl.random_su3_field(dims, 22)
        Ug = _gauge_transform(U, g)
        psi = wl.random_spinor(dims, 23)
        gpsi = np.einsum("...ab,...sb->...sa", g, psi)
        A, Ag = oracle.clover_matrix(U, kappa, csw), oracle.clover_matrix(Ug, kappa, csw)
        lhs = oracle.apply_D(Ug, Ag, bc, kappa, gpsi)
        rhs = np.einsum("...ab,...sb->...sa", g, oracle.apply_D(U, A, bc, kappa, psi))
        assert np.abs(lhs - rhs).max() / np.abs(rhs).max() < 1e-13
        # clover alone transforms by conjugation
        assert np.abs(oracle.site_matvec(Ag, gpsi) - np.einsum("...ab,...sb->...sa", g, oracle.site_matvec(A, psi))).max() < 1e-13


def test_P5_abelian_clover_closed_form():
    """Links diag(e^{i th}, e^{-i th}, 1): (Fhat_{mu nu})_11 = (i/4) sum of sin(plaquette angle) over the
    four plaquettes touching x in the (mu,nu) plane, _22 = minus that, _33 = 0."""
    dims = (4, 6, 4, 8)
    X, Y, Z, T = dims
    rng = np.random.default_rng(31)
    th = rng.uniform(-np.pi, np.pi, size=(4, T, Z, Y, X))
    U = np.zeros((4, T, Z, Y, X, 3, 3), dtype=complex)
    U[..., 0, 0] = np.exp(1j * th)
    U[..., 1, 1] = np.exp(-1j * th)
    U[..., 2, 2] = 1
    F = oracle.fhat(U)
    ax = lambda m: 3 - m
    planes = [(0, 1), (0, 2), (0, 3), (1, 2), (1, 3), (2, 3)]
    for pl, (mu, nu) in enumerate(planes):
        P = th[mu] + np.roll(th[nu], -1, axis=ax(mu)) - np.roll(th[mu], -1, axis=ax(nu)) - th[nu]
        S = np.sin(P)
        tot = S + np.roll(S, 1, axis=ax(mu)) + np.roll(np.roll(S, 1, axis=ax(mu)), 1, axis=ax(nu)) + np.roll(S, 1, axis=ax(nu))
        assert np.abs(F[pl][..., 0, 0] - 0.25j * tot).max() < 1e-14
        assert np.abs(F[pl][..., 1, 1] + 0.25j * tot).max() < 1e-14
        assert np.abs(F[pl][..., 2, 2]).max() < 1e-14
        off = F[pl].copy()
        off[..., [0, 1, 2], [0, 1, 2]] = 0
        assert np.abs(off).max() < 1e-14


def test_P6_tree_level_improvement():
    """c_sw = +1 must cancel the O(a) term: with N the naive operator, D(c_sw)/(2 kappa) at kappa = 1/8
    equals N - N^2/2 up to O(a^2) only for c_sw = 1.  A wrong sign doubles the error, c_sw = 0 leaves it."""
    L = 16
    dims = (L, L, L, L)
    bc = (1, 1, 1, 1)
    kappa = 1.0 / 8.0
    rng = np.random.default_rng(41)
    t, z, y, x = np.meshgrid(*[np.arange(L)] * 4, indexing="ij")
    coords = [x, y, z, t]
    # smooth algebra fields: for each direction mu and generator a, a sum of 3 low cosines
    U = np.empty((4, L, L, L, L, 3, 3), dtype=complex)
    for mu in range(4):
        f = np.zeros((8, L, L, L, L))
        for a in range(8):
            for _ in range(3):
                k = rng.integers(-1, 2, size=4)
                f[a] += rng.standard_normal() * np.cos(2 * np.pi * sum(k[m] * coords[m] for m in range(4)) / L + rng.uniform(0, 2 * np.pi))
        H = np.einsum("a...,aij->...ij", f, wl._GM) / 2
        U[mu] = wl.expi(H.reshape(-1, 3, 3), 0.1).reshape(L, L, L, L, 3, 3)
    n = (1, -1, 0, 1)
    p = 2 * np.pi * np.array(n) / L
    u = rng.standard_normal((4, 3)) + 1j * rng.standard_normal((4, 3))
    psi = _plane_wave(dims, p)[..., None, None] * u

    def naive(v):
        out = np.zeros_like(v)
        for mu in range(4):
            a = 3 - mu
            fwd = np.einsum("...ab,...sb->...sa", U[mu], np.roll(v, -1, axis=a))
            bwd = np.roll(np.einsum("...ba,...sb->...sa", U[mu].conj(), v), 1, axis=a)
            out += 0.5 * np.einsum("st,...tc->...sc", GAMMA[mu], fwd - bwd)
        return out

    Npsi = naive(psi)
    target = Npsi - 0.5 * naive(Npsi)
    err = {}
    for c in (1.0, 0.0, -1.0):
        A = oracle.clover_matrix(U, kappa, c)
        Dm = oracle.apply_D(U, A, bc, kappa, psi) / (2 * kappa)
        err[c] = np.linalg.norm(Dm - target) / np.linalg.norm(target)
    assert err[1.0] < 0.5 * err[0.0]
    assert 1.7 < err[-1.0] / err[0.0] < 2.3


def test_P7_clover_structure():
    dims, kappa, csw = (4, 4, 4, 8), 0.118, 1.5
    U = wl.gauge_links(dims, 0.4, 51)
    A = oracle.clover_matrix(U, kappa, csw)
    assert np.abs(A - np.conj(np.swapaxes(A, -1, -2))).max() < 1e-15
    assert np.abs(A[..., :6, 6:]).max() == 0.0 and np.abs(A[..., 6:, :6]).max() == 0.0
    G5 = np.kron(GAMMA5, np.eye(3))
    assert np.abs(A @ G5 - G5 @ A).max() == 0.0
    # definition re-assembled from Fhat and the sigma matrices typed in tests/gammas.py
    F = oracle.fhat(U)
    planes = [(0, 1), (0, 2), (0, 3), (1, 2), (1, 3), (2, 3)]
    B = np.broadcast_to(np.eye(12, dtype=complex), A.shape).copy()
    for pl, (mu, nu) in enumerate(planes):
        B += 1j * csw * kappa * np.einsum("st,...ab->...satb", sigma(mu, nu), F[pl]).reshape(A.shape)
    assert np.abs(A - B).max() < 1e-15
    # Fhat anti-Hermitian
    assert np.abs(F + np.conj(np.swapaxes(F, -1, -2))).max() < 1e-15
    Ainv = oracle.clover_inverse(A)
    assert np.abs(Ainv @ A - np.eye(12)).max() < 1e-13
    assert np.abs(Ainv - np.linalg.inv(A)).max() < 1e-13


@pytest.mark.parametrize("eps,plaq", [(0.2, 0.899), (0.3, 0.785), (0.4, 0.647), (0.5, 0.503)])
def test_link_generator_plaquette(eps, plaq):
    """Sanity pin of the input recipe: unitarity, det = 1, average plaquette."""
    dims = (8, 8, 8, 8)
    U = wl.gauge_links(dims, eps, 61)
    assert np.abs(U @ np.conj(np.swapaxes(U, -1, -2)) - np.eye(3)).max() < 1e-13
    assert np.abs(np.linalg.det(U) - 1).max() < 1e-13
    tot, cnt = 0.0, 0
    for mu in range(4):
        for nu in range(mu + 1, 4):
            a, b = 3 - mu, 3 - nu
            P = U[mu] @ np.roll(U[nu], -1, axis=a) @ np.conj(np.swapaxes(np.roll(U[mu], -1, axis=b), -1, -2)) @ np.conj(np.swapaxes(U[nu], -1, -2))
            tot += np.trace(P, axis1=-2, axis2=-1).real.mean() / 3
            cnt += 1
    assert abs(tot / cnt - plaq) < 0.004
