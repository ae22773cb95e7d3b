"""P4 (BASELINE.json north_star check 4): on a 2^4 lattice build D densely, invert it by Gauss-Jordan,
and check (a) the oracle's BiCGStab against D^{-1} eta, (b) the stochastic estimator of PAPER.md eq. 7.3
(L300) S ~ (1/(N_r scale^2)) sum_r psi_r eta_r^dagger, whose error falls as 1/sqrt(N_r):
for iid unit-modulus noise E||S_hat - S||_F^2 = ((n-1)/N_r) ||S||_F^2 exactly, n = 192."""
import numpy as np
import pytest

import oracle
from paper_1405_4524_b200 import workloads as wl

DIMS = (2, 2, 2, 2)
BC = (1, 1, 1, -1)
KAPPA, CSW = 0.120, 1.0


@pytest.fixture(scope="module")
def dense():
    U = wl.gauge_links(DIMS, 0.3, 71)
    A = oracle.clover_matrix(U, KAPPA, CSW)
    M = oracle.dense_D(U, A, BC, KAPPA)
    S = oracle.dense_inverse(M)
    return U, A, M, S


def test_dense_matrix_is_the_operator(dense):
    U, A, M, S = dense
    x = wl.random_spinor(DIMS, 72)
    assert np.abs(M @ x.ravel() - oracle.apply_D(U, A, BC, KAPPA, x).ravel()).max() < 1e-14
    assert np.abs(S @ M - np.eye(192)).max() < 1e-13
    assert np.abs(S - np.linalg.inv(M)).max() < 1e-12           # library inverse as a second opinion
    # gamma5-hermiticity of the dense matrix: (G5 M)^dagger = G5 M
    g5 = np.tile(np.repeat([1, 1, -1, -1], 3), 16)
    G5M = g5[:, None] * M
    assert np.abs(G5M - G5M.conj().T).max() < 1e-14


def test_bicgstab_equals_dense_inverse(dense):
    U, A, M, S = dense
    eta = oracle.noise_fill(DIMS, 2001, 3, scale=wl.INV_SQRT2)
    for r in range(3):
        psi, info = oracle.bicgstab(U, A, BC, KAPPA, eta[r], tol=1e-13)
        assert info["status"] == 0 and info["true_resid"] < 1e-12
        want = S @ eta[r].ravel()
        assert np.linalg.norm(psi.ravel() - want) / np.linalg.norm(want) < 1e-11


@pytest.mark.parametrize("scale", [1.0, wl.INV_SQRT2])
def test_estimator_variance_scaling(dense, scale):
    U, A, M, S = dense
    n = 192
    nmax = 1024
    eta = oracle.noise_fill(DIMS, 2001, nmax, scale=scale).reshape(nmax, n)
    psi = eta @ S.T                                              # psi_r = D^{-1} eta_r
    S2 = np.linalg.norm(S) ** 2
    ratios = []
    for nr in (16, 64, 256, 1024):
        # average the squared error over independent groups of nr sources (fewer groups as nr grows)
        errs = []
        for g in range(nmax // nr):
            sl = slice(g * nr, (g + 1) * nr)
            Shat = psi[sl].T @ eta[sl].conj() / (nr * scale * scale)
            errs.append(np.linalg.norm(Shat - S) ** 2)
        ratios.append(np.mean(errs) * nr / ((n - 1) * S2))
    assert all(0.9 < r < 1.1 for r in ratios), ratios
    # the N_r = 64 case BASELINE.json configs[1] names: relative error is O(1), not small
    Shat = psi[:64].T @ eta[:64].conj() / (64 * scale * scale)
    rel = np.linalg.norm(Shat - S) / np.linalg.norm(S)
    assert 1.4 < rel < 2.1
    if scale != 1.0:
        # without the 1/scale^2 the estimator converges to scale^2 * S, not S (DESIGN R7)
        Sraw = psi.T @ eta.conj() / nmax
        assert np.linalg.norm(Sraw - scale ** 2 * S) < np.linalg.norm(Sraw - S)
