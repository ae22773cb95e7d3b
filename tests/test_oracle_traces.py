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
