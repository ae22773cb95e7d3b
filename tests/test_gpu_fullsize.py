"""GPU parity at BASELINE.json's full sizes, in the launch configuration bench.py times (cfg 3: 24^3x48, batch 8, mixed;
cfg 4: 32^3x64, two-row links, time dilution).  The oracle cannot solve these in seconds, so: (a) the fused operators are
compared element by element on whole fields (one oracle D apply ~ 1 s), (b) every checked GPU solution gets an
oracle-computed true residual, (c) solution parity is checked through the property psi = D^-1 eta <=> D psi = eta with the
oracle's D, which pins psi to the unique solution within cond(D) * 1e-10."""
import numpy as np
import pytest
import torch

import oracle
from paper_1405_4524_b200 import workloads as wl

pytestmark = pytest.mark.gpu


def _run(ci, n_solve, check):
    from paper_1405_4524_b200 import binding as B
    c = wl.CONFIGS[ci]
    dims = c["dims"]
    U = wl.gauge_links(dims, c["eps"], c["gauge_seed"])
    A = oracle.clover_matrix(U, c["kappa"], c["csw"])
    ctx = B.Clover(torch.from_numpy(U).cuda(), c["kappa"], c["csw"], bc=wl.BC, recon=c["recon"], max_rhs=8)
    # sources of the first and the last batch of the config (cfg 4: timeslices 0.. and ..63)
    first = B.noise_fill(dims, c["noise_seed"], n_solve, rhs_offset=0, time_dilution=c["dilution"], scale=wl.INV_SQRT2)
    last = B.noise_fill(dims, c["noise_seed"], n_solve, rhs_offset=c["n_rhs"] - n_solve, time_dilution=c["dilution"], scale=wl.INV_SQRT2)
    want = oracle.noise_fill(dims, c["noise_seed"], 1, rhs_offset=c["n_rhs"] - 1, time_dilution=c["dilution"], scale=wl.INV_SQRT2)
    assert np.array_equal(last[-1].cpu().numpy().view(np.uint64), want[0].view(np.uint64))        # noise bit-exact at full size
    # operators on whole fields, fp64 and fp32 (the batch-8 kernels)
    x = first.cpu().numpy()
    ref = oracle.apply_D(U, A, wl.BC, c["kappa"], x[0])
    got = ctx.dslash_apply(B.OP_D_FULL, first)[0].cpu().numpy()
    assert np.abs(got - ref).max() / np.abs(ref).max() < 1e-13
    got32 = ctx.dslash_apply(B.OP_D_FULL, first.to(torch.complex64))[0].cpu().numpy()
    assert np.abs(got32 - ref).max() / np.abs(ref).max() < 1e-6
    hop = oracle.hop(U, wl.BC, x[0])
    got32 = ctx.dslash_apply(B.OP_HOP_FULL, first.to(torch.complex64))[0].cpu().numpy()
    assert np.abs(got32 - hop).max() / np.abs(hop).max() < 1e-6
    del got, got32, ref, hop
    for eta in (first, last):
        psi, infos, bad = ctx.solve(eta, tol=wl.TOL, batch=c["batch"], mixed=bool(c["mixed"]))
        assert bad == 0, infos
        e, p = eta.cpu().numpy(), psi.cpu().numpy()
        for r in check:
            res = np.linalg.norm(e[r] - oracle.apply_D(U, A, wl.BC, c["kappa"], p[r])) / np.linalg.norm(e[r])
            assert res <= wl.TOL, (r, res)
            assert abs(infos[r]["true_resid"] - res) <= 1e-3 * res + 1e-14
    ctx.close()


def test_cfg3_24x24x24x48_batch8_mixed():
    _run(3, 8, check=(0, 7))


def test_cfg4_32x32x32x64_recon12_dilution():
    _run(4, 8, check=(7,))
