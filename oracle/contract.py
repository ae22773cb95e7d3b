"""oracle/contract.py -- TEST INFRASTRUCTURE, NOT THE PRODUCT (see oracle/__init__.py).

Plain numpy statement of the stochastic-operator contraction of arXiv:1405.4524, eqs. 7.5-7.7:

    O_ij(t)   = sum_y eta_i^*(t, y) gamma5 X_j(t, y)                       (7.6)   sum over space, spin, colour
    C(t - t0) = N_r^-2 sum_ij Tr[ O_ij(t) O_ji(t0) ]                       (7.7)

eta_i are the noise sources, X_j = D^-1 eta_j the solution vectors (layout [n, T, Z, Y, X, 4, 3] complex128, spin index
in the basis of DESIGN.md R1 where gamma5 = diag(+1, +1, -1, -1)).  O_ij(t) is a complex number per (t, i, j); the "Tr" of
(7.7) is then the plain product.  With noise of variance scale^2 each propagator estimate S ~ (1/(N_r scale^2)) sum X eta^+
(R7) carries 1/scale^2, so the correlator is divided by scale^4.  Pins: tests/test_oracle_contract.py.
"""
import numpy as np

GAMMA5 = np.array([1.0, 1.0, -1.0, -1.0])


def stochastic_operators(eta, X):
    """O[t, i, j] = sum_{z,y,x,s,c} conj(eta[i,t,z,y,x,s,c]) gamma5[s] X[j,t,z,y,x,s,c]   (eq. 7.6)."""
    eta = np.asarray(eta, dtype=np.complex128)
    X = np.asarray(X, dtype=np.complex128)
    g5X = X * GAMMA5[:, None]
    return np.einsum("itzyxsc,jtzyxsc->tij", eta.conj(), g5X)


def correlator(O, scale=1.0):
    """C[t0, t] = (1 / (N_r^2 scale^4)) sum_ij O[t, i, j] O[t0, j, i]   (eq. 7.7, every pair of timeslices)."""
    n = O.shape[1]
    return np.einsum("tij,uji->ut", O, O) / (n * n * scale ** 4)
