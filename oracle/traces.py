"""oracle/traces.py -- TEST INFRASTRUCTURE, NOT THE PRODUCT (see oracle/__init__.py).

The two trace operations of Table I of arXiv:1405.4524, per timeslice t:

    sum_y     Tr[ S_p(t,y; 0,0) S_p^dagger(t,y; 0,0) ]           S_p = the 12 point-source solutions (spin-colour columns)
    sum_x,z   Tr[ S_s(t,z; 0,x) S_s^dagger(t,z; 0,x) ]           S_s = the filled stochastic propagator (oracle/fill.py)

"the dagger is only w.r.t. the spin-color indices", so both are the squared Frobenius norm of everything that
lives on timeslice t: out[t] = sum_{o, k} |f[o, t, k]|^2 for a field viewed as [n_outer, T, slice_len].
By gamma5-hermiticity the first one is the zero-momentum pion correlator sum_y Tr[S(t,y;0,0) g5 S(0,0;t,y) g5] (pinned).
"""
import numpy as np


def timeslice_norm2(f, n_outer, T):
    f = np.asarray(f, dtype=np.complex128).reshape(n_outer, T, -1)
    return np.sum(f.real ** 2 + f.imag ** 2, axis=(0, 2))


def timeslice_inner(a, b, n_outer, T):
    """out[t] = sum_{o, k} a[o, t, k] conj(b[o, t, k]): with a, b two fills of eq. 7.3 from INDEPENDENT source sets this is
    sum_x sum_z Tr[S_s^(1)(t,z;0,x) S_s^(2)dagger(t,z;0,x)], the paper's "two sets of random sources, one for S and one for
    S^dagger", whose point (Figs. 2-3) is that it has no noise-squared bias; a = b gives timeslice_norm2."""
    a = np.asarray(a, dtype=np.complex128).reshape(n_outer, T, -1)
    b = np.asarray(b, dtype=np.complex128).reshape(n_outer, T, -1)
    return np.sum(a * np.conj(b), axis=(0, 2))
