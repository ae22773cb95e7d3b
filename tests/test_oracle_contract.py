"""Pins for the oracle of the stochastic-operator contraction (eqs. 7.5-7.7).  CPU only."""
import numpy as np

import oracle
from oracle import contract
from gammas import GAMMA5
from paper_1405_4524_b200 import workloads as wl


def test_brute_force_loops_on_a_tiny_lattice():
    dims, n = (2, 2, 2, 4), 3
    X_, Y_, Z_, T_ = dims
    eta = wl.random_spinor(dims, 1, n)
    X = wl.random_spinor(dims, 2, n)
    g5 = np.diag(GAMMA5).real                      # independently typed gamma5 (tests/gammas.py)
    want = np.zeros((T_, n, n), dtype=complex)
    for t in range(T_):
        for i in range(n):
            for j in range(n):
                acc = 0
                for z in range(Z_):
                    for y in range(Y_):
                        for x in range(X_):
                            for s in range(4):
                                for c in range(3):
                                    acc += np.conj(eta[i, t, z, y, x, s, c]) * g5[s] * X[j, t, z, y, x, s, c]
                want[t, i, j] = acc
    got = contract.stochastic_operators(eta, X)
    assert np.abs(got - want).max() < 1e-13
    C = contract.correlator(got, scale=0.5)
    for t0 in range(T_):
        for t in range(T_):
            w = sum(want[t, i, j] * want[t0, j, i] for i in range(n) for j in range(n)) / (n * n * 0.5 ** 4)
            assert abs(C[t0, t] - w) < 1e-12 * max(1, abs(w))


def test_identity_propagator_special_case():
    """X = eta (S = 1): O_ji = conj(O_ij) because gamma5 is Hermitian, and O_ii(t) = scale^2 L^3 tr(gamma5 (x) 1) = 0 exactly."""
    dims = (4, 4, 2, 4)
    eta = oracle.noise_fill(dims, 5, 6, scale=wl.INV_SQRT2)
    O = contract.stochastic_operators(eta, eta)
    assert np.abs(O - np.conj(np.swapaxes(O, 1, 2))).max() < 1e-13
    assert np.abs(np.einsum("tii->ti", O)).max() < 1e-13
    # linearity in X and antilinearity in eta
    X = wl.random_spinor(dims, 3, 6)
    assert np.allclose(contract.stochastic_operators(2j * eta, 3 * X), -2j * 3 * contract.stochastic_operators(eta, X))


def test_correlator_estimates_the_exact_trace_on_2x2x2x4():
    """On a lattice small enough for the dense inverse (the paper's own validation strategy):
    the off-diagonal (i != j) part of eq. 7.7 is an unbiased estimator of sum_{x,y} Tr[S(t0,x;t,y) g5 S(t,y;t0,x) g5]."""
    dims, kappa, csw, bc = (2, 2, 2, 4), 0.12, 1.0, (1, 1, 1, -1)
    X_, Y_, Z_, T_ = dims
    U = wl.gauge_links(dims, 0.3, 81)
    A = oracle.clover_matrix(U, kappa, csw)
    S = oracle.dense_inverse(oracle.dense_D(U, A, bc, kappa))          # [n, n], n = 12 V, index ((t z y x) s c)
    V3 = X_ * Y_ * Z_
    nt = 12 * V3
    G5 = np.tile(np.repeat([1.0, 1.0, -1.0, -1.0], 3), V3)
    exact = np.zeros((T_, T_), dtype=complex)                          # exact[t0, t]
    for t0 in range(T_):
        for t in range(T_):
            S01 = S[t0 * nt:(t0 + 1) * nt, t * nt:(t + 1) * nt]        # S(t0, x; t, y)
            S10 = S[t * nt:(t + 1) * nt, t0 * nt:(t0 + 1) * nt]        # S(t, y; t0, x)
            exact[t0, t] = np.trace(S01 @ (G5[:, None] * S10) * G5[None, :])
    n, scale = 1500, wl.INV_SQRT2
    eta = oracle.noise_fill(dims, 2001, n, scale=scale)
    X = (eta.reshape(n, -1) @ S.T).reshape(eta.shape)                   # X_r = D^-1 eta_r
    O = contract.stochastic_operators(eta, X)
    full = np.einsum("tij,uji->ut", O, O)
    diag = np.einsum("tii,uii->ut", O, O)
    est = (full - diag) / (n * (n - 1) * scale ** 4)
    assert np.abs(est - exact).max() / np.abs(exact).max() < 0.05
    # the paper's formula with all pairs differs from it only by the O(1/N_r) diagonal terms
    assert np.abs(contract.correlator(O, scale) - est).max() / np.abs(exact).max() < 0.1
    # and the zero-momentum pion correlator is real and positive: Tr[S g5 S g5] = ||S(t,.;t0,.)||_F^2 by g5-hermiticity
    assert np.abs(exact.imag).max() < 1e-12 and exact.real.min() > 0
