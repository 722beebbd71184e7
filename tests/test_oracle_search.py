"""End-to-end pins for the oracle: an independent numpy/scipy route on tiny inputs, injection recovery, false alarms."""
import numpy as np
import pytest
from scipy import special, stats

from paper_2406_15186_b200 import synth


def library_route(spec, zmax, B, C, thr, n_trials=1.0, widths=None):
    """The same path through library routines only (numpy.median, scipy MAD, cumsum differences, chi2.logsf,
    norm.isf) — slow, tiny inputs."""
    n = spec.size
    nb = max(1, n // B)
    P = np.empty(n)
    for j in range(nb):
        lo, hi = j * B, (n if j == nb - 1 else (j + 1) * B)
        comps = []
        for v in (spec.real[lo:hi].astype(np.float64), spec.imag[lo:hi].astype(np.float64)):
            s = stats.median_abs_deviation(v, scale="normal")
            comps.append((v - np.median(v)) / s if s > 0 else np.zeros_like(v))
        P[lo:hi] = 0.5 * (comps[0] ** 2 + comps[1] ** 2)
    pre = np.concatenate([[0.0], np.cumsum(P)])
    out = []
    for c in range((n + C - 1) // C):
        lo, hi = c * C, min((c + 1) * C, n)
        best = None
        for w in (range(1, zmax + 1) if widths is None else widths):
            i = np.arange(lo, min(hi, n - w + 1))
            if i.size == 0:
                continue
            S = pre[i + w] - pre[i]
            k = int(np.argmax(S))
            lnp = min(0.0, stats.chi2.logsf(2 * S[k], 2 * w) + np.log(n_trials))
            if best is None or lnp < best[0]:
                best = (lnp, int(i[k]), w, S[k])
        if best is not None and best[0] <= special.log_ndtr(-thr):
            out.append((best[1], best[2], best[3], stats.norm.isf(np.exp(best[0]))))
    return out


@pytest.mark.parametrize("seed,n,zmax,B,C,thr", [(0, 257, 8, 64, 16, 2.0), (1, 513, 20, 128, 20, 2.5),
                                                  (2, 300, 12, 512, 7, 1.5), (3, 1025, 16, 256, 64, 3.0)])
def test_search_matches_library_route(orc, seed, n, zmax, B, C, thr):
    rng = np.random.default_rng(seed)
    spec = (rng.normal(0, 30, n) + 1j * rng.normal(0, 30, n)).astype(np.complex64)
    spec[n // 3: n // 3 + 5] *= 4.0  # a bump so that something is significant
    got = orc.search(spec, zmax, B, C, thr)
    ref = library_route(spec, zmax, B, C, thr)
    assert len(got) == len(ref) > 0
    for g, r in zip(got, ref):
        assert (g["bin"], g["width"]) == (r[0], r[1])
        assert g["power"] == pytest.approx(r[2], rel=1e-11)
        assert g["sigma"] == pytest.approx(r[3], abs=1e-7)
    # sorted by bin, at most one per block, bin inside its block
    assert np.all(np.diff(got["bin"] // C) > 0)


def test_searched_width_sets_follow_the_paper(orc):
    # L411: "only search logarithmically spaced (i.e. z = 1, 2, 4, 8, ... z-max)"; width = z + 1 (R9); z = 0 kept (R28)
    assert [w for w in range(1, 41) if orc.width_searched(w, log_sampling=True)] == [1, 2, 3, 5, 9, 17, 33]
    # Alg. 4: z from 0, searched when remainder(z / z_step) = 0
    assert [w for w in range(1, 15) if orc.width_searched(w, z_step=4)] == [1, 5, 9, 13]
    assert all(orc.width_searched(w) for w in range(1, 100))                       # default: every width (north_star)
    assert [w for w in range(1, 12) if orc.width_searched(w, z_step=3, log_sampling=True)] == [1, 2, 3, 5, 9]  # log wins


@pytest.mark.parametrize("z_step,log_sampling", [(1, False), (3, False), (7, False), (1, True)])
def test_sampled_search_matches_library_route(orc, z_step, log_sampling):
    n, zmax, B, C, thr = 769, 24, 256, 32, 2.0
    rng = np.random.default_rng(11)
    spec = (rng.normal(0, 30, n) + 1j * rng.normal(0, 30, n)).astype(np.complex64)
    spec[200:212] *= 2.5
    spec[500:503] *= 4.0
    if log_sampling:
        widths = [w for w in range(1, zmax + 1) if w == 1 or (w - 1) & (w - 2) == 0]     # z = w − 1 ∈ {0} ∪ powers of two
    else:
        widths = [w for w in range(1, zmax + 1) if (w - 1) % z_step == 0]
    got = orc.search(spec, zmax, B, C, thr, z_step=z_step, log_sampling=log_sampling)
    ref = library_route(spec, zmax, B, C, thr, widths=widths)
    assert len(got) == len(ref) > 0
    assert set(got["width"].tolist()) <= set(widths)
    for g, r in zip(got, ref):
        assert (g["bin"], g["width"]) == (r[0], r[1])
        assert g["power"] == pytest.approx(r[2], rel=1e-11)
        assert g["sigma"] == pytest.approx(r[3], abs=1e-7)
    if z_step == 1 and not log_sampling:
        assert np.array_equal(got, orc.search(spec, zmax, B, C, thr))


def test_r_block_reports_block_index_times_width(orc):
    # L222-226: "simply saving the block index"; Table 3: R-Block r = 360448 = 11 x 32768 for the exact r = 364318
    assert 364318 // 32768 * 32768 == 360448
    n, zmax, B, C, thr = 2049, 16, 512, 100, 2.5
    rng = np.random.default_rng(5)
    spec = (rng.normal(0, 30, n) + 1j * rng.normal(0, 30, n)).astype(np.complex64)
    spec[700:706] *= 4.0
    exact = orc.search(spec, zmax, B, C, thr)
    approx = orc.search(spec, zmax, B, C, thr, r_block=True)
    assert len(exact) == len(approx) > 0
    assert np.array_equal(approx["bin"], exact["bin"] // C * C)
    for f in ("spectrum", "width", "power", "sigma"):
        assert np.array_equal(approx[f], exact[f])


def test_per_width_emission_is_every_block_width_above_threshold(orc):
    # Alg. 4: one candidate per (chunk, searched z); L322: the highest sigma one is picked afterwards
    n, zmax, B, C, thr = 1025, 12, 256, 64, 2.5
    rng = np.random.default_rng(21)
    spec = (rng.normal(0, 30, n) + 1j * rng.normal(0, 30, n)).astype(np.complex64)
    spec[300:306] *= 3.5
    allw = orc.search_harmonics(spec, zmax, B, C, thr, 1, per_width=True)
    best = orc.search(spec, zmax, B, C, thr)
    M, I = orc.block_maxima(orc.normalise_power(spec, B), zmax, C)
    want = []
    for c in range(M.shape[0]):
        for w in range(1, zmax + 1):
            if I[c, w - 1] >= 0 and stats.chi2.logsf(2 * M[c, w - 1], 2 * w) <= special.log_ndtr(-thr):
                want.append((int(I[c, w - 1]), w))
    assert list(zip(allw["bin"].tolist(), allw["width"].tolist())) == want and len(want) > len(best)
    for r in best:                                             # the default output = the highest-sigma record of each block
        mine = allw[allw["bin"] // C == r["bin"] // C]
        top = mine[np.argmax(mine["sigma"])]
        assert (top["bin"], top["width"]) == (r["bin"], r["width"]) and top["sigma"] == r["sigma"]


def test_bonferroni_trials_shift(orc):
    rng = np.random.default_rng(4)
    spec = (rng.normal(0, 1, 600) + 1j * rng.normal(0, 1, 600)).astype(np.complex64)
    spec[100:104] *= 6
    a = orc.search(spec, 8, 128, 32, 3.0, n_trials=1.0)
    b = orc.search(spec, 8, 128, 32, 3.0, n_trials=50.0)
    ref = library_route(spec, 8, 128, 32, 3.0, n_trials=50.0)
    assert len(b) == len(ref) <= len(a)
    for g, r in zip(b, ref):
        assert (g["bin"], g["width"]) == (r[0], r[1]) and g["sigma"] == pytest.approx(r[3], abs=1e-7)


def test_batch_rows_are_independent(orc):
    rng = np.random.default_rng(5)
    specs = (rng.normal(0, 9, (3, 2049)) + 1j * rng.normal(0, 9, (3, 2049))).astype(np.complex64)
    specs[1, 700:712] *= 3
    full = orc.search(specs, 16, 512, 64, 3.0)
    for b in range(3):
        alone = orc.search(specs[b], 16, 512, 64, 3.0)
        sub = full[full["spectrum"] == b]
        assert np.array_equal(alone["bin"], sub["bin"]) and np.array_equal(alone["width"], sub["width"])
        assert np.array_equal(alone["sigma"], sub["sigma"])   # bit-exact


def test_pitch_larger_than_n_bins(orc):
    rng = np.random.default_rng(6)
    specs = (rng.normal(0, 9, (2, 1100)) + 1j * rng.normal(0, 9, (2, 1100))).astype(np.complex64)
    a = orc.search(specs, 8, 256, 50, 2.5, n_bins=1025)
    b = orc.search(np.ascontiguousarray(specs[:, :1025]), 8, 256, 50, 2.5)
    assert np.array_equal(a, b)


def test_config1_injection_is_recovered(orc):
    # BASELINE config 1: 2^16 samples, 173.2 Hz, A = 0.05, z = 12; zmax 32, B 1024, C 64, σ ≥ 6.
    wl = synth.CONFIGS[1]
    X, inj = synth.make_spectra(wl)
    cands = orc.search(X.numpy(), wl.zmax, wl.norm_block, wl.block_width, wl.sigma_threshold)
    assert len(cands) >= 1
    top = cands[np.argmax(cands["sigma"])]
    start = inj[0].expected_start_bin(wl.t_obs)            # 726.45
    assert abs(top["bin"] - start) <= 4
    assert abs(top["width"] - (abs(inj[0].z) + 1)) <= 0.25 * (abs(inj[0].z) + 1) + 1   # width tracks |z|+1
    assert top["sigma"] >= 6.5
    # frozen fixture values (oracle output for seed 2; regenerate only with a cited reason)
    assert (int(top["bin"]), int(top["width"])) == (727, 14)
    assert top["sigma"] == pytest.approx(7.065, abs=2e-3)


@pytest.mark.parametrize("z,amp,f0", [(20.0, 0.05, 310.7), (-60.0, 0.06, 97.3), (90.0, 0.07, 411.9)])
def test_width_tracks_drift(orc, z, amp, f0):
    # scaled-down config-2-like case: 2^19 samples, one chirp; width ≈ |z|+1 loosely (Table 2: gradient 0.78)
    wl = synth.CONFIGS[2].scaled(n_samples=1 << 19, zmax=100, norm_block=2048, block_width=100, n_fixed_random=0,
                                 fixed=(synth.Injection(0, f0, amp, z),), seed=77)
    X, inj = synth.make_spectra(wl)
    cands = orc.search(X.numpy(), wl.zmax, wl.norm_block, wl.block_width, 6.0)
    top = cands[np.argmax(cands["sigma"])]
    start = inj[0].expected_start_bin(wl.t_obs)
    assert abs(top["bin"] - start) <= 6
    assert 0.6 * (abs(z) + 1) <= top["width"] <= 1.35 * (abs(z) + 1)
    assert top["sigma"] > 8


def test_noise_only_false_alarm_count(orc):
    # ≤ n·zmax·sf(thr) expected per spectrum (an upper bound: overlapping windows are correlated); at thr = 4 that is
    # 2^17 · 32 · 3.2e-5 ≈ 133, and far more than zero.
    rng = np.random.default_rng(8)
    n = (1 << 17) + 1
    spec = (rng.normal(0, 100, n) + 1j * rng.normal(0, 100, n)).astype(np.complex64)
    cands = orc.search(spec, 32, 2048, 64, 4.0)
    bound = n * 32 * stats.norm.sf(4.0)
    assert 5 < len(cands) < 1.3 * bound
    assert len(orc.search(spec, 32, 2048, 64, 7.0)) == 0
