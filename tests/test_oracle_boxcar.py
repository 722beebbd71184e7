"""Pins for the oracle's boxcar sums and per-block maxima (§2.2.5; Alg. 4)."""
import numpy as np
import pytest


def brute_sums(P, zmax):
    """O(n·zmax) direct definition: S(i,w) = Σ_{j<w} P[i+j]."""
    n = P.size
    out = np.full((zmax, n), np.nan)
    for w in range(1, zmax + 1):
        for i in range(0, n - w + 1):
            out[w - 1, i] = sum(P[i + j] for j in range(w))
    return out


@pytest.mark.parametrize("n,zmax", [(1, 1), (5, 5), (17, 6), (40, 12), (64, 64)])
def test_recursion_equals_brute_force_and_prefix_differences(orc, n, zmax):
    rng = np.random.default_rng(n + zmax)
    P = rng.exponential(size=n)
    S = orc.boxcar_sums(P, zmax)
    B = brute_sums(P, zmax)
    assert np.array_equal(np.isnan(S), np.isnan(B))
    np.testing.assert_allclose(np.nan_to_num(S), np.nan_to_num(B), rtol=1e-13)
    pre = np.concatenate([[0.0], np.cumsum(P)])
    for w in range(1, zmax + 1):
        np.testing.assert_allclose(S[w - 1, : n - w + 1], pre[w:] - pre[:-w], rtol=1e-12)


def test_output_length_is_n_minus_w_plus_1(orc):
    # "Output length N-1", "N-2"
    S = orc.boxcar_sums(np.ones(10), 4)
    for w in range(1, 5):
        assert np.isfinite(S[w - 1]).sum() == 10 - w + 1


def test_ramp_closed_form(orc):
    # X = [1..N]: S(i,w) = w(i+1) + w(w-1)/2 (0-based i)
    N, zmax = 50, 9
    S = orc.boxcar_sums(np.arange(1, N + 1, dtype=float), zmax)
    for w in range(1, zmax + 1):
        i = np.arange(N - w + 1)
        assert np.array_equal(S[w - 1, : N - w + 1], w * (i + 1) + w * (w - 1) / 2)


def test_paper_worked_example_y2_y3(orc):
    # Y2 = [x1+x2, x2+x3, ...], Y3 = Y2[:end-1] + X[3:end]
    x = np.array([3.0, 1.0, 4.0, 1.0, 5.0, 9.0])
    S = orc.boxcar_sums(x, 3)
    assert np.array_equal(S[1, :5], x[:-1] + x[1:])
    assert np.array_equal(S[2, :4], S[1, :4] + x[2:])


def test_sums_monotone_in_width_for_nonnegative_power(orc):
    rng = np.random.default_rng(3)
    S = orc.boxcar_sums(rng.exponential(size=100), 20)
    for w in range(1, 20):
        valid = np.isfinite(S[w])
        assert np.all(S[w][valid] >= S[w - 1][valid])


@pytest.mark.parametrize("n,zmax,C", [(30, 7, 8), (64, 16, 16), (65, 10, 16), (100, 25, 7), (9, 12, 4)])
def test_block_maxima_match_brute_force(orc, n, zmax, C):
    rng = np.random.default_rng(n * zmax + C)
    P = rng.exponential(size=n)
    M, I = orc.block_maxima(P, zmax, C)
    B = brute_sums(P, zmax)
    nblk = (n + C - 1) // C
    assert M.shape == (nblk, zmax)
    for c in range(nblk):
        lo, hi = c * C, min((c + 1) * C, n)
        for w in range(1, zmax + 1):
            vals = B[w - 1, lo:hi]
            ok = np.isfinite(vals)
            if not ok.any():           # no window of this width starts in the block (R11)
                assert M[c, w - 1] == -1 and I[c, w - 1] == -1
                continue
            assert M[c, w - 1] == pytest.approx(np.nanmax(vals), rel=1e-13)
            assert I[c, w - 1] == lo + int(np.nanargmax(vals))


def test_ties_pick_lowest_bin(orc):
    P = np.zeros(32)
    P[[3, 5, 19]] = 7.0  # equal spikes: in block 0 (bins 0-15) the lowest bin attaining the max must win (R14)
    M, I = orc.block_maxima(P, 2, 16)
    assert I[0, 0] == 3 and I[1, 0] == 19
    assert I[0, 1] == 2  # width 2: windows starting at 2,3,4,5 all sum to 7 → lowest start


def test_window_belongs_to_block_of_its_first_bin(orc):
    # R12 / Alg. 4: the halo is read from the next chunk; moving a spike across the boundary moves the owner
    P = np.full(64, 0.1)
    P[16] = 50.0                       # first bin of block 1 (C = 16)
    M, I = orc.block_maxima(P, 4, 16)
    assert I[1, 0] == 16 and M[1, 0] == 50.0
    assert I[0, 0] != 16               # width 1: block 0 does not see it
    assert I[0, 1] == 15 and M[0, 1] == pytest.approx(50.1)   # width 2 starting at bin 15 reaches into block 1
    P2 = np.full(64, 0.1)
    P2[15] = 50.0
    M2, I2 = orc.block_maxima(P2, 4, 16)
    assert I2[0, 0] == 15 and M2[1, 0] == pytest.approx(0.1)
