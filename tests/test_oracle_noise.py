"""P8: pins for the Z4 noise of the oracle (docs/NOISE.md)."""
import os

import numpy as np

import oracle
from paper_1405_4524_b200 import workloads as wl


def test_splitmix64_published_vectors():
    assert [oracle.splitmix64(0, c) for c in range(3)] == [0xE220A8397B1DCDAF, 0x6E789E6AA1B965F4, 0x06C45D188009454F]
    golden = os.path.join(os.path.dirname(__file__), "golden", "splitmix64_seed1234567.txt")
    want = [int(line) for line in open(golden) if line.strip() and not line.startswith("#")]
    assert len(want) == 5 and [oracle.splitmix64(1234567, c) for c in range(5)] == want


def test_noise_matches_spec_in_python_ints():
    """Re-derive k from the spec with Python integers at scattered (r, site, s, c)."""
    dims = (4, 6, 2, 8)
    X, Y, Z, T = dims
    V = X * Y * Z * T
    seed, off = 2000, 3
    eta = oracle.noise_fill(dims, seed, 2, rhs_offset=off, scale=1.0)
    M = (1 << 64) - 1
    z4 = [1, 1j, -1, -1j]
    rng = np.random.default_rng(0)
    for _ in range(200):
        j, t, z, y, x, s, c = [int(rng.integers(0, m)) for m in (2, T, Z, Y, X, 4, 3)]
        n = (((t * Z + z) * Y + y) * X + x) * 12 + 3 * s + c
        ctr = (off + j) * 12 * V + n
        v = (seed + 0x9E3779B97F4A7C15 * (ctr + 1)) & M
        v = ((v ^ (v >> 30)) * 0xBF58476D1CE4E5B9) & M
        v = ((v ^ (v >> 27)) * 0x94D049BB133111EB) & M
        v ^= v >> 31
        assert eta[j, t, z, y, x, s, c] == z4[v >> 62]


def test_noise_statistics_and_bits():
    dims = (8, 8, 8, 16)
    s = wl.INV_SQRT2
    eta = oracle.noise_fill(dims, 2001, 4, scale=s)
    re, im = eta.real, eta.imag
    assert np.all((np.abs(re) == s) ^ (np.abs(im) == s))          # unit modulus * scale, one part exactly zero
    assert not np.signbit(re[re == 0]).any() and not np.signbit(im[im == 0]).any()   # zeros are +0.0
    n = eta.size
    for v in (s, 1j * s, -s, -1j * s):
        f = np.count_nonzero(eta == v) / n
        assert abs(f - 0.25) < 4 * np.sqrt(0.25 * 0.75 / n)
    # independent sources are uncorrelated: |<eta_a, eta_b>| / n ~ 1/sqrt(n)
    c = abs(np.vdot(eta[0], eta[1])) / (s * s * eta[0].size)
    assert c < 5 / np.sqrt(eta[0].size)
    # fp32 variant: same k, float-rounded scale
    eta32 = oracle.noise_fill(dims, 2001, 4, scale=s, dtype=np.float32)
    assert np.array_equal(np.sign(eta32.real), np.sign(re)) and np.array_equal(np.sign(eta32.imag), np.sign(im))
    assert set(np.unique(np.abs(eta32.real))) == {np.float32(0), np.float32(s)}


def test_noise_time_dilution_is_a_mask():
    dims = (4, 4, 4, 8)
    full = oracle.noise_fill(dims, 2004, 10, rhs_offset=5, scale=1.0)
    dil = oracle.noise_fill(dims, 2004, 10, rhs_offset=5, time_dilution=1, scale=1.0)
    for j in range(10):
        tr = (5 + j) % 8
        assert np.array_equal(dil[j, tr], full[j, tr])
        rest = np.delete(dil[j], tr, axis=0)
        assert np.all(rest == 0) and not np.signbit(rest.real).any() and not np.signbit(rest.imag).any()
    # rhs_offset only shifts the stream
    a = oracle.noise_fill(dims, 7, 3, rhs_offset=0, scale=1.0)
    b = oracle.noise_fill(dims, 7, 1, rhs_offset=2, scale=1.0)
    assert np.array_equal(a[2], b[0])


def test_spin_colour_dilution_masks_and_covers():
    """dilution bits (docs/NOISE.md; "time-spin-color dilution"): each source is a masked copy of its undiluted
    stream, and 12 T consecutive time-spin-colour diluted sources touch every (t, spin, colour) exactly once."""
    dims = (2, 2, 2, 4)
    T = 4
    n = 12 * T
    full = oracle.noise_fill(dims, 9, n, scale=1.0)
    tsc = oracle.noise_fill(dims, 9, n, scale=1.0, dilution=3)
    sc_only = oracle.noise_fill(dims, 9, 24, scale=1.0, dilution=2)
    cover = np.zeros((T, 4, 3), dtype=int)
    for r in range(n):
        t_r, sc_r = r % T, (r // T) % 12
        mask = np.zeros(full[r].shape, dtype=bool)
        mask[t_r, :, :, :, sc_r // 3, sc_r % 3] = True
        assert np.array_equal(tsc[r][mask], full[r][mask]) and np.all(tsc[r][~mask] == 0)
        assert not np.signbit(tsc[r].real).any() or np.all(tsc[r].real[np.signbit(tsc[r].real)] != 0)
        cover[t_r, sc_r // 3, sc_r % 3] += 1
    assert np.all(cover == 1)
    for r in range(24):
        sc_r = r % 12
        mask = np.zeros(full[r].shape, dtype=bool)
        mask[:, :, :, :, sc_r // 3, sc_r % 3] = True
        assert np.array_equal(sc_only[r][mask], full[r][mask]) and np.all(sc_only[r][~mask] == 0)
