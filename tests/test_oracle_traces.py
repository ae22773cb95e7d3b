"""Pins for the oracle of the Table I trace operations.  CPU only."""
import numpy as np

import oracle
from oracle import traces, fill
from paper_1405_4524_b200 import workloads as wl


def test_brute_force_and_total():
    rng = np.random.default_rng(0)
    f = rng.standard_normal((3, 4, 10)) + 1j * rng.standard_normal((3, 4, 10))
    got = traces.timeslice_norm2(f, 3, 4)
    for t in range(4):
        assert abs(got[t] - sum(abs(f[o, t, k]) ** 2 for o in range(3) for k in range(10))) < 1e-12
    assert abs(got.sum() - np.linalg.norm(f) ** 2) < 1e-11


def test_point_source_trace_is_the_pion_correlator():
    """sum_y Tr[S S^dagger](t) from the 12 exact point-source columns equals sum_y Tr[S(t,y;0,0) g5 S(0,0;t,y) g5] computed from
    OTHER entries of the dense inverse (gamma5-hermiticity)."""
    dims, kappa, csw, bc = (2, 2, 2, 4), 0.12, 1.0, (1, 1, 1, -1)
    U = wl.gauge_links(dims, 0.3, 93)
    A = oracle.clover_matrix(U, kappa, csw)
    S = oracle.dense_inverse(oracle.dense_D(U, A, bc, kappa))
    nt = 12 * 8
    cols = S[:, :12]                                   # source at (t, z, y, x) = 0, the 12 spin-colour columns
    Sp = cols.T.reshape(12, 4, nt)                     # [column, t, (site, a)] = the 12 "solution vectors"
    got = traces.timeslice_norm2(Sp, 12, 4)
    g5 = np.repeat([1.0, 1.0, -1.0, -1.0], 3)
    for t in range(4):
        want = 0
        for y in range(8):
            fwd = S[t * nt + 12 * y: t * nt + 12 * y + 12, :12]        # S(t,y; 0,0)
            bwd = S[:12, t * nt + 12 * y: t * nt + 12 * y + 12]        # S(0,0; t,y)
            want += np.trace(fwd @ (g5[:, None] * bwd) * g5[None, :])
        assert abs(want.imag) < 1e-12 and abs(got[t] - want.real) < 1e-12 * abs(want.real) + 1e-14


def test_stochastic_trace_is_the_norm_of_the_fill():
    dims = (2, 2, 2, 4)
    X = wl.random_spinor(dims, 3, 5)
    eta = wl.random_spinor(dims, 4, 5)
    S = fill.stochastic_fill(X, eta, t0=1)
    got = traces.timeslice_norm2(S, 1, 4)
    for t in range(4):
        assert abs(got[t] - np.linalg.norm(S[t]) ** 2) < 1e-10


def test_inner_brute_force_and_symmetries():
    rng = np.random.default_rng(1)
    a = rng.standard_normal((2, 3, 7)) + 1j * rng.standard_normal((2, 3, 7))
    b = rng.standard_normal((2, 3, 7)) + 1j * rng.standard_normal((2, 3, 7))
    c = rng.standard_normal((2, 3, 7)) + 1j * rng.standard_normal((2, 3, 7))
    got = traces.timeslice_inner(a, b, 2, 3)
    for t in range(3):
        assert abs(got[t] - sum(a[o, t, k] * np.conj(b[o, t, k]) for o in range(2) for k in range(7))) < 1e-12
    assert np.abs(traces.timeslice_inner(b, a, 2, 3) - np.conj(got)).max() < 1e-12                       # Hermitian form
    assert np.abs(traces.timeslice_inner(a + 2j * c, b, 2, 3) - got - 2j * traces.timeslice_inner(c, b, 2, 3)).max() < 1e-11
    nn = traces.timeslice_inner(a, a, 2, 3)
    assert np.abs(nn.imag).max() < 1e-13 and np.abs(nn.real - traces.timeslice_norm2(a, 2, 3)).max() < 1e-12
    assert abs(got.sum() - np.vdot(b, a)) < 1e-11


def test_one_set_is_biased_two_independent_sets_are_not():
    """The paper's lesson (Figs. 2-3) in closed form.  With S_hat = S P, P = (1/N) sum eta eta^+ over N iid
    unit-modulus sources on the n = 12 L^3 source components, E[P] = 1 and E[P P^+] = (1 + (n-1)/N) 1, so the one-set trace
    sum Tr[S_hat S_hat^+](t) overshoots the exact sum_x sum_z Tr[S S^+](t) by the factor 1 + (n-1)/N, while the trace between
    fills from two independent sets, sum Tr[S_hat1 S_hat2^+](t), is unbiased."""
    dims, kappa, csw, bc, t0, scale = (2, 2, 2, 4), 0.12, 1.0, (1, 1, 1, -1), 0, wl.INV_SQRT2
    U = wl.gauge_links(dims, 0.3, 94)
    A = oracle.clover_matrix(U, kappa, csw)
    Sx = oracle.dense_inverse(oracle.dense_D(U, A, bc, kappa))
    nt, n = 12 * 8, 400
    exact = traces.timeslice_norm2(Sx[:, t0 * nt:(t0 + 1) * nt].reshape(4, nt * nt), 1, 4)
    fills = []
    for seed in (3001, 3002):
        eta = oracle.noise_fill(dims, seed, n, scale=scale)
        eta[:, np.arange(4) != t0] = 0                                  # sources on timeslice t0 only (time dilution)
        psi = (eta.reshape(n, -1) @ Sx.T).reshape(eta.shape)
        fills.append(fill.stochastic_fill(psi, eta, t0=t0, scale=scale))
    one = traces.timeslice_norm2(fills[0], 1, 4)
    two = traces.timeslice_inner(fills[0], fills[1], 1, 4)
    assert np.abs(one / (exact * (1 + (nt - 1) / n)) - 1).max() < 0.05
    assert np.abs(two.real / exact - 1).max() < 0.05 and np.abs(two.imag / exact).max() < 0.05
    assert np.all(one / exact > 1.15)                                    # the bias is there: (n-1)/N = 0.24
