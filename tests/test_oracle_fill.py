"""Pins for the oracle of the outer-product fill (eq. 7.3).  CPU only."""
import numpy as np

import oracle
from oracle import fill
from paper_1405_4524_b200 import workloads as wl


def test_brute_force_loops():
    dims, n, t0, scale = (2, 2, 2, 4), 3, 1, 0.5
    X = wl.random_spinor(dims, 1, n)
    eta = wl.random_spinor(dims, 2, n)
    S = fill.stochastic_fill(X, eta, t0=t0, scale=scale)
    Sd = fill.stochastic_fill(X, eta, t0=t0, scale=scale, dagger=True)
    rng = np.random.default_rng(0)
    for _ in range(300):
        t, z, y, x, s, c = [int(rng.integers(0, m)) for m in (4, 2, 2, 2, 4, 3)]
        z2, y2, x2, s2, c2 = [int(rng.integers(0, m)) for m in (2, 2, 2, 4, 3)]
        want = sum(X[i, t, z, y, x, s, c] * np.conj(eta[i, t0, z2, y2, x2, s2, c2]) for i in range(n)) / (n * scale ** 2)
        z3, x3 = (z * 2 + y) * 2 + x, (z2 * 2 + y2) * 2 + x2
        assert abs(S[t, z3, 3 * s + c, x3, 3 * s2 + c2] - want) < 1e-13
        assert abs(Sd[x3, 3 * s2 + c2, t, z3, 3 * s + c] - np.conj(want)) < 1e-13


def test_fill_is_the_estimator_of_the_dense_inverse():
    """The paper's validation (L39-41, L303): on a lattice with an exact inverse, the fill is the block of columns at t0 of
    S_hat = (1/(N_r scale^2)) sum psi eta^+ and converges to D^-1 there as 1/sqrt(N_r) with the exactly known variance."""
    dims, kappa, csw, bc, t0, scale = (2, 2, 2, 4), 0.12, 1.0, (1, 1, 1, -1), 2, wl.INV_SQRT2
    U = wl.gauge_links(dims, 0.3, 91)
    A = oracle.clover_matrix(U, kappa, csw)
    Sx = oracle.dense_inverse(oracle.dense_D(U, A, bc, kappa))               # index ((t z y x) s c), 384 x 384
    n = 2000
    eta = oracle.noise_fill(dims, 2001, n, scale=scale)
    psi = (eta.reshape(n, -1) @ Sx.T).reshape(eta.shape)
    got = fill.stochastic_fill(psi, eta, t0=t0, scale=scale)                  # [t, z3, a, x3, b]
    nt = 12 * 8
    full = psi.reshape(n, -1).T @ eta.reshape(n, -1).conj() / (n * scale ** 2)   # the estimator written as one matrix product
    assert np.abs(got.reshape(4 * nt, nt) - full[:, t0 * nt:(t0 + 1) * nt]).max() < 1e-12
    exact = Sx[:, t0 * nt:(t0 + 1) * nt]
    # exact expectation for iid unit-modulus noise: E||S_hat - S||^2 over the column block = (n_t ||S||_F^2 - ||S_block||_F^2) / N_r
    ratio = np.linalg.norm(got.reshape(4 * nt, nt) - exact) ** 2 * n / (nt * np.linalg.norm(Sx) ** 2 - np.linalg.norm(exact) ** 2)
    assert 0.9 < ratio < 1.1
