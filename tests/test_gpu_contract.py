"""GPU parity of the stochastic-operator contraction (paper eqs. 7.5-7.7) against oracle/contract.py: element by element,
1e-13 scale-normalised (fp64, reading R9).  Sizes span several (i, j) tiles, ragged tiles, ragged k-chunks."""
import numpy as np
import pytest
import torch

import oracle
from oracle import contract
from paper_1405_4524_b200 import workloads as wl

pytestmark = pytest.mark.gpu


def nerr(got, want):
    return np.abs(got - want).max() / np.abs(want).max()


@pytest.mark.parametrize("dims,n", [((4, 4, 4, 8), 5), ((4, 6, 2, 4), 32), ((2, 2, 2, 2), 40), ((6, 4, 4, 6), 70), ((8, 8, 8, 16), 16)])
def test_operators_and_correlator(dims, n):
    from paper_1405_4524_b200 import binding as B
    eta = wl.random_spinor(dims, 11, n)
    X = wl.random_spinor(dims, 12, n)
    want = contract.stochastic_operators(eta, X)
    o = B.stochastic_operators(torch.from_numpy(eta).cuda(), torch.from_numpy(X).cuda())
    got = o.cpu().numpy()
    assert got.shape == want.shape and nerr(got, want) < 1e-13
    wc = contract.correlator(want, scale=wl.INV_SQRT2)
    gc = B.stochastic_correlator(o, scale=wl.INV_SQRT2).cpu().numpy()
    assert nerr(gc, wc) < 1e-12


def test_pipeline_noise_solve_contract():
    """noise_fill -> clover_solve -> stochastic_operators on the device against the oracle's contraction of the same fields,
    and the pion correlator it gives is real and positive up to noise (gamma5-hermiticity)."""
    from paper_1405_4524_b200 import binding as B
    c = wl.CONFIGS[0]
    dims = c["dims"]
    U = wl.gauge_links(dims, c["eps"], c["gauge_seed"])
    ctx = B.Clover(torch.from_numpy(U).cuda(), c["kappa"], c["csw"], bc=wl.BC, max_rhs=8)
    eta = B.noise_fill(dims, c["noise_seed"], 24, scale=wl.INV_SQRT2)
    psi, infos, bad = ctx.solve(eta, tol=wl.TOL, batch=8, mixed=True)
    assert bad == 0
    o = B.stochastic_operators(eta, psi)
    want = contract.stochastic_operators(eta.cpu().numpy(), psi.cpu().numpy())
    assert nerr(o.cpu().numpy(), want) < 1e-13
    C = B.stochastic_correlator(o, scale=wl.INV_SQRT2).cpu().numpy()
    assert np.all(np.diag(C).real > 0)          # t = t0: dominated by the contact term ||S(t,.;t,.)||^2
    ctx.close()


def test_full_size_cfg3_sampled_timeslices():
    """24^3x48, N_r = 32 (the bench configuration of the contraction): timeslices 0, 17 and 47 against the oracle."""
    from paper_1405_4524_b200 import binding as B
    dims, n = wl.CONFIGS[3]["dims"], 32
    eta = B.noise_fill(dims, 2003, n, scale=wl.INV_SQRT2)
    X = B.noise_fill(dims, 977, n, scale=1.0)                       # any field serves as X for the contraction itself
    X = X * torch.linspace(0.5, 1.5, n, device="cuda", dtype=torch.float64).view(n, 1, 1, 1, 1, 1, 1)
    o = B.stochastic_operators(eta, X).cpu().numpy()
    for t in (0, 17, 47):
        want = contract.stochastic_operators(eta[:, t:t + 1].cpu().numpy(), X[:, t:t + 1].cpu().numpy())[0]
        assert nerr(o[t], want) < 1e-13
