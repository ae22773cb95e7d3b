"""Host-side check of the algebra behind the merged BiCGStab ordering of csrc/solver.cu (step 3).

The CUDA solver moves the dot products of the textbook recurrence so that BLAS-1 traffic rides in the Dslash
epilogues.  The identities it relies on are exact-arithmetic statements about ANY gamma5-hermitian operator (M^+ = G M G):

    <r0, M p>  = <q0, p>            with q0 = M^+ r0 = G M G r0        (alpha known before M p is applied)
    rho'       = <r0, s> - omega <r0, t>                                (= <r0, r'> with r' = s - omega t)
    p'         = r' + beta p - gam (r - s),  gam = rho'/rho             (r - s = alpha v, beta omega / alpha = rho'/rho)

Both orderings are written out here in numpy fp64 on a small dense gamma5-hermitian matrix and must produce the same iterates.
Nothing here touches oracle/ or the CUDA path; it pins the formulas the kernels implement (SC_OMEGA2 / SC_RHO2 / xrp_update_kernel).
"""
import numpy as np


def _system(n=48, seed=5):
    rng = np.random.default_rng(seed)
    G = np.diag(np.where(np.arange(n) < n // 2, 1.0, -1.0))
    H = rng.normal(size=(n, n)) + 1j * rng.normal(size=(n, n))
    H = (H + H.conj().T) / np.sqrt(8 * n)
    M = np.eye(n) + 0.6 * G @ H          # M^+ = 1 + 0.6 H G = G M G
    assert np.allclose(M.conj().T, G @ M @ G)
    b = rng.normal(size=n) + 1j * rng.normal(size=n)
    return M, G, b


def _dot(a, b):
    return np.vdot(a, b)   # sum conj(a) b


def textbook(M, b, iters):
    x = np.zeros_like(b); r = b.copy(); r0 = r.copy(); p = r.copy(); rho = _dot(r0, r)
    out = []
    for _ in range(iters):
        v = M @ p
        alpha = rho / _dot(r0, v)
        s = r - alpha * v
        t = M @ s
        omega = _dot(t, s) / _dot(t, t)
        x = x + alpha * p + omega * s
        r = s - omega * t
        rho1 = _dot(r0, r)
        beta = (rho1 / rho) * (alpha / omega)
        p = r + beta * (p - omega * v)
        rho = rho1
        out.append((x.copy(), r.copy(), p.copy()))
    return out


def merged(M, G, b, iters):
    x = np.zeros_like(b); r = b.copy(); r0 = r.copy(); p = r.copy()
    q0 = G @ (M @ (G @ r0))                      # restart: q0 = M^+ r0
    rho = _dot(r, r); alpha = rho / _dot(q0, p)  # SC_RESTART2
    out = []
    for _ in range(iters):
        s = r - alpha * (M @ p)                  # Dslash epilogue DOT_S: v is never stored
        t = M @ s                                # Dslash epilogue DOT_XW: <t,s>, <t,t>, <r0,t>, <r0,s>
        omega = _dot(t, s) / _dot(t, t)          # SC_OMEGA2
        rho1 = _dot(r0, s) - omega * _dot(r0, t)
        gam = rho1 / rho
        beta = gam * (alpha / omega)
        rho = rho1
        x = x + alpha * p + omega * s            # xrp_update_kernel
        rn = s - omega * t
        p = rn + beta * p - gam * (r - s)
        r = rn
        alpha = rho / _dot(q0, p)                # SC_RHO2
        out.append((x.copy(), r.copy(), p.copy()))
    return out


def test_merged_ordering_reproduces_the_textbook_iterates():
    M, G, b = _system()
    a, c = textbook(M, b, 12), merged(M, G, b, 12)
    for k, ((xa, ra, pa), (xc, rc, pc)) in enumerate(zip(a, c)):
        scale = np.linalg.norm(b)
        assert np.linalg.norm(xa - xc) <= 1e-11 * np.linalg.norm(xa), k
        assert np.linalg.norm(ra - rc) <= 1e-11 * scale and np.linalg.norm(pa - pc) <= 1e-11 * scale, k
    # and both solve the system
    x = c[-1][0]
    assert np.linalg.norm(b - M @ x) / np.linalg.norm(b) < 1e-6


def test_identities_one_by_one():
    M, G, b = _system(seed=11)
    rng = np.random.default_rng(3)
    r0, p = (rng.normal(size=b.size) + 1j * rng.normal(size=b.size) for _ in range(2))
    q0 = G @ (M @ (G @ r0))
    assert abs(_dot(r0, M @ p) - _dot(q0, p)) < 1e-12 * np.linalg.norm(r0) * np.linalg.norm(p)
    # alpha chosen from <q0,p> makes s orthogonal to r0, which is why rho' is dominated by -omega <r0,t>
    r = b
    alpha = _dot(r0, r) / _dot(q0, p)
    s = r - alpha * (M @ p)
    assert abs(_dot(r0, s)) < 1e-12 * np.linalg.norm(r0) * np.linalg.norm(r)
    # a frozen right-hand side (alpha = omega = beta = gam = 0) is a fixed point of the sweep: x, r unchanged, p = r
    x = rng.normal(size=b.size) + 0j
    s0 = r - 0 * (M @ p)
    assert np.array_equal(x + 0 * p + 0 * s0, x) and np.array_equal(s0 - 0 * (M @ s0), r) and np.array_equal((s0 - 0 * (M @ s0)) + 0 * p - 0 * (r - s0), r)
