"""oracle/fill.py -- TEST INFRASTRUCTURE, NOT THE PRODUCT (see oracle/__init__.py).

Plain numpy statement of the stochastic all-to-all estimator of arXiv:1405.4524, eq. 7.3:

    S(t, z; t0, x) ~ (1 / N_r) sum_i X_i(t, z) eta_i^*(t0, x)

("S_s fill", 12 x 12 x T x L^3 x L^3 entries; the dagger version "S_s^dagger fill" stores the Hermitian
conjugate).  With noise of variance scale^2 the estimator carries 1/scale^2 (R7).
Layouts: X, eta complex128 [n, T, Z, Y, X, 4, 3];  S[t, z3, a, x3, b] with z3, x3 = flattened (z, y, x) spatial sites and
a, b = 3*spin + colour;  S_dagger[x3, b, t, z3, a] = conj(S[t, z3, a, x3, b]).  Pins: tests/test_oracle_fill.py.
"""
import numpy as np


def stochastic_fill(X, eta, t0=0, scale=1.0, dagger=False):
    X = np.asarray(X, dtype=np.complex128)
    eta = np.asarray(eta, dtype=np.complex128)
    n, T = X.shape[0], X.shape[1]
    V3 = X.shape[2] * X.shape[3] * X.shape[4]
    Xf = X.reshape(n, T, V3, 12)
    e0 = eta[:, t0].reshape(n, V3, 12)
    S = np.einsum("itza,ixb->tzaxb", Xf, e0.conj()) / (n * scale * scale)
    return np.conj(np.transpose(S, (3, 4, 0, 1, 2))) if dagger else S
