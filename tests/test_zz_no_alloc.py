"""GPU test of the allocation-free entry point stochastic_operators_noalloc (include/clover.h; paper eq. 7.6) against
the existing path stochastic_operators, element by element at the 1e-13 scale-normalised tolerance of tests/test_gpu_contract.py.
Collected last on purpose (file name): the suite runs with `pytest -x`, so a failure here must not hide the other tests.

Two calls in a row share the library's fixed scratch array, which keeps the first call's contents: the second call uses other inputs and
another shape (fewer sources, so part of the first call's partial sums is still in the array behind its own), and a third call repeats the
first shape.  The oracle (oracle/contract.py) is checked on the first call as well, so the test stands on its own in a fresh process."""
import numpy as np
import pytest
import torch

from oracle import contract
from paper_1405_4524_b200 import workloads as wl

pytestmark = pytest.mark.gpu

TOL = 1e-13   # tests/test_gpu_contract.py: max|gpu - oracle| / max|oracle|


def nerr(got, want):
    return np.abs(got - want).max() / np.abs(want).max()


def _pair(B, dims, n, seed):
    eta = torch.from_numpy(wl.random_spinor(dims, seed, n)).cuda()
    x = torch.from_numpy(wl.random_spinor(dims, seed + 1, n)).cuda()
    T = dims[3]
    out = torch.full((T, n, n), float("nan"), dtype=torch.complex128, device="cuda")   # caller-owned output, poisoned
    return eta, x, out


def test_noalloc_matches_existing_path_on_consecutive_calls():
    from paper_1405_4524_b200 import binding as B
    dims = (4, 6, 4, 8)
    calls = [(40, 301), (9, 311), (40, 321)]        # (n_rhs, seed): ragged 32 x 32 tiles, then a smaller problem, then the first shape again
    for k, (n, seed) in enumerate(calls):
        eta, x, out = _pair(B, dims, n, seed)
        want = B.stochastic_operators(eta, x).cpu().numpy()                 # existing path (cudaMallocAsync scratch)
        free_before = torch.cuda.mem_get_info()[0]
        got = B.stochastic_operators_noalloc(eta, x, out)
        torch.cuda.synchronize()
        assert torch.cuda.mem_get_info()[0] >= free_before                  # the call took no device memory (a pool may have released some)
        got = got.cpu().numpy()
        assert np.isfinite(got).all() and nerr(got, want) < TOL, (k, nerr(got, want))
        if k == 0:
            ref = contract.stochastic_operators(eta.cpu().numpy(), x.cpu().numpy())
            assert nerr(got, ref) < TOL


def test_noalloc_twice_on_the_same_inputs_is_bit_identical_and_sizes_are_checked():
    from paper_1405_4524_b200 import binding as B
    dims = (8, 8, 8, 16)
    eta, x, out1 = _pair(B, dims, 32, 401)
    out2 = torch.full_like(out1, float("nan"))
    want = B.stochastic_operators(eta, x)
    B.stochastic_operators_noalloc(eta, x, out1)
    B.stochastic_operators_noalloc(eta, x, out2)                            # second call in a row on the same stream: ordered, no race
    torch.cuda.synchronize()
    assert torch.equal(out1, out2)
    assert nerr(out1.cpu().numpy(), want.cpu().numpy()) < TOL
    # beyond the fixed scratch: T * n^2 = 16 * 260^2 > NOALLOC_MAX_TNN -> a clear error, nothing launched
    small = (2, 2, 2, 16)
    n_big = 260
    assert small[3] * n_big * n_big > B.NOALLOC_MAX_TNN
    e_big = torch.zeros((n_big, 16, 2, 2, 2, 4, 3), dtype=torch.complex128, device="cuda")
    o_big = torch.zeros((16, n_big, n_big), dtype=torch.complex128, device="cuda")
    with pytest.raises(B.CloverError, match="exceeds"):
        B.stochastic_operators_noalloc(e_big, e_big, o_big)
    # ... and exactly at the limit it runs: T * n^2 = 16 * 256^2 = NOALLOC_MAX_TNN (one k-chunk)
    n_lim = 256
    e_lim = torch.from_numpy(wl.random_spinor(small, 411, n_lim)).cuda()
    o_lim = torch.empty((16, n_lim, n_lim), dtype=torch.complex128, device="cuda")
    B.stochastic_operators_noalloc(e_lim, e_lim, o_lim)
    assert nerr(o_lim.cpu().numpy(), B.stochastic_operators(e_lim, e_lim).cpu().numpy()) < TOL
