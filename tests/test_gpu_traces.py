"""GPU parity of the Table I trace operations against oracle/traces.py (fp64, 1e-13), and the paper's validation on its own
4^3x8 lattice: the pion correlator from 12 point-source solves against the stochastic one from the filled propagator."""
import numpy as np
import pytest
import torch

import oracle
from oracle import traces
from paper_1405_4524_b200 import workloads as wl

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("n_outer,T,L", [(1, 4, 7), (12, 8, 768), (3, 16, 100003), (2, 2, 1)])
def test_timeslice_norm2(n_outer, T, L):
    from paper_1405_4524_b200 import binding as B
    rng = np.random.default_rng(5)
    f = rng.standard_normal((n_outer, T, L)) + 1j * rng.standard_normal((n_outer, T, L))
    got = B.timeslice_norm2(torch.from_numpy(f).cuda(), n_outer, T).cpu().numpy()
    want = traces.timeslice_norm2(f, n_outer, T)
    assert np.abs(got - want).max() / np.abs(want).max() < 1e-13


@pytest.mark.parametrize("n_outer,T,L", [(1, 4, 7), (12, 8, 768), (3, 16, 100003), (2, 2, 1)])
def test_timeslice_inner(n_outer, T, L):
    from paper_1405_4524_b200 import binding as B
    rng = np.random.default_rng(6)
    a = rng.standard_normal((n_outer, T, L)) + 1j * rng.standard_normal((n_outer, T, L))
    b = rng.standard_normal((n_outer, T, L)) + 1j * rng.standard_normal((n_outer, T, L))
    ad, bd = torch.from_numpy(a).cuda(), torch.from_numpy(b).cuda()
    got = B.timeslice_inner(ad, bd, n_outer, T).cpu().numpy()
    want = traces.timeslice_inner(a, b, n_outer, T)
    scale = np.sqrt(traces.timeslice_norm2(a, n_outer, T) * traces.timeslice_norm2(b, n_outer, T)).max()
    assert np.abs(got - want).max() / scale < 1e-13
    same = B.timeslice_inner(ad, ad, n_outer, T).cpu().numpy()
    assert np.abs(same.imag).max() == 0.0 and np.abs(same.real - traces.timeslice_norm2(a, n_outer, T)).max() / scale < 1e-13


def test_point_and_stochastic_pion_correlators_on_4x4x4x8():
    """compare stochastic propagators with exact point-source ones on a lattice small enough.  The whole
    pipeline runs on the device: 12 point solves -> sum_y Tr S_p S_p^+ ; noise -> solves -> fill -> sum_x sum_z Tr S_s S_s^+."""
    from paper_1405_4524_b200 import binding as B
    c = wl.CONFIGS[0]
    dims = c["dims"]
    X, Y, Z, T = dims
    V3 = X * Y * Z
    U = wl.gauge_links(dims, c["eps"], c["gauge_seed"])
    ctx = B.Clover(torch.from_numpy(U).cuda(), c["kappa"], c["csw"], bc=wl.BC, max_rhs=8)
    src = torch.zeros((12, T, Z, Y, X, 4, 3), dtype=torch.complex128, device="cuda")
    for s in range(4):
        for col in range(3):
            src[3 * s + col, 0, 0, 0, 0, s, col] = 1
    Sp, infos, bad = ctx.solve(src, tol=wl.TOL, batch=4, mixed=True)
    assert bad == 0
    Cp = B.timeslice_norm2(Sp, 12, T).cpu().numpy()
    assert np.abs(Cp - traces.timeslice_norm2(Sp.cpu().numpy(), 12, T)).max() / Cp.max() < 1e-13
    # the oracle's own point propagator (one column) agrees with ours, so Cp is the exact correlator of this configuration
    A = oracle.clover_matrix(U, c["kappa"], c["csw"])
    ref, _ = oracle.bicgstab(U, A, wl.BC, c["kappa"], src[5].cpu().numpy(), tol=1e-12)
    assert np.linalg.norm(Sp[5].cpu().numpy() - ref) / np.linalg.norm(ref) < 1e-8
    # stochastic: N_r sources, fill at t0 = 0, trace; E|S_hat|^2 = |S|^2 + variance, so subtract the known noise floor:
    # E||S_hat[t]||_F^2 = ||S[t, :, cols at t0]||_F^2 + (n_t ||S[t]||^2_rows... ) -- here only the 1/N_r trend is checked
    n = 512
    eta = B.noise_fill(dims, c["noise_seed"], n, scale=wl.INV_SQRT2)
    psi, infos, bad = ctx.solve(eta, tol=wl.TOL, batch=8, mixed=True)
    assert bad == 0
    Cs = {}
    for m in (128, 512):
        S = B.stochastic_fill(psi[:m].contiguous(), eta[:m].contiguous(), t0=0, scale=wl.INV_SQRT2)
        Cs[m] = B.timeslice_norm2(S, 1, T).cpu().numpy() / V3          # average over the source position x
        assert np.abs(Cs[m] - traces.timeslice_norm2(S.cpu().numpy(), 1, T) / V3).max() / Cs[m].max() < 1e-13
    # ||S_hat||^2 = signal + noise/N_r: two N_r values separate them; the signal must have the size and fall-off of the exact
    # point-source correlator (source-position average vs the origin: agreement to a few 10 % on this rough configuration)
    signal = (512 * Cs[512] - 128 * Cs[128]) / (512 - 128)
    assert np.all(signal > 0)
    assert 0.5 < signal[0] / Cp[0] < 2.0 and 0.3 < signal[T // 2] / Cp[T // 2] < 3.0
    assert Cp[0] > Cp[1] > Cp[2] and signal[0] > signal[1] > signal[2]
    # the paper's other option (L303, Figs. 2-3): S and S^+ from two independent source sets -- no noise floor to subtract
    S1 = B.stochastic_fill(psi[:256].contiguous(), eta[:256].contiguous(), t0=0, scale=wl.INV_SQRT2)
    S2 = B.stochastic_fill(psi[256:].contiguous(), eta[256:].contiguous(), t0=0, scale=wl.INV_SQRT2)
    two = B.timeslice_inner(S1, S2, 1, T).cpu().numpy() / V3
    want = traces.timeslice_inner(S1.cpu().numpy(), S2.cpu().numpy(), 1, T) / V3
    assert np.abs(two - want).max() / np.abs(want).max() < 1e-12
    for t in range(3):
        assert 0.6 < two[t].real / signal[t] < 1.6 and abs(two[t].imag) < 0.3 * signal[t]
        assert Cs[128][t] > 2 * two[t].real          # the one-set trace carries the (n-1)/N_r noise-squared bias
    ctx.close()
