"""Pins for the oracle's harmonic sum (§2.3): closed form, a numpy reshape route, the χ² degrees of
freedom the paper states, the search through library routines, and the point of the method (harmonics add up)."""
import numpy as np
import pytest
from scipy import special, stats


def reshape_route(P, H):
    """Y_H from non-overlapping group sums by reshape (library route): D_h = group sums of h, truncated to floor(n/H)."""
    nH = P.size // H
    Y = np.zeros(nH)
    for h in range(1, H + 1):
        m = P.size // h
        Y += P[: m * h].reshape(m, h).sum(axis=1)[:nH]
    return Y


@pytest.mark.parametrize("n,H", [(12, 1), (12, 2), (13, 3), (29, 4), (1000, 4), (7, 4)])
def test_harmonic_sum_ramp_closed_form_and_reshape(orc, n, H):
    P = np.arange(1, n + 1, dtype=np.float64)
    Y = orc.harmonic_sum(P, H)
    assert Y.size == n // H                                             # complete groups only (R29)
    r = np.arange(n // H, dtype=np.float64)
    # D_h(r) = sum_{j<h} (h r + j + 1) = h^2 r + h(h+1)/2
    closed = sum(h * h * r + h * (h + 1) / 2 for h in range(1, H + 1))
    assert np.array_equal(Y, closed)
    rng = np.random.default_rng(n + H)
    Q = rng.exponential(size=n)
    assert np.allclose(orc.harmonic_sum(Q, H), reshape_route(Q, H), rtol=1e-14, atol=0)


@pytest.mark.parametrize("H", [2, 3, 4])
def test_harmonic_sum_degrees_of_freedom(orc, H):
    # L214-216: X_H ~ chi^2(sum_{n<=H} 2n) = chi^2(H(H+1)); in mean-1 units a Gamma variate of shape H(H+1)/2
    rng = np.random.default_rng(100 + H)
    P = rng.exponential(size=400_000)
    Y = orc.harmonic_sum(P, H)
    kappa = H * (H + 1) / 2
    assert Y.mean() == pytest.approx(kappa, rel=5e-3)
    # neighbouring bins of Y_H share inputs only through different h, so thin before the KS test
    assert stats.kstest(Y[:: 4 * H], stats.gamma(kappa).cdf).pvalue > 1e-3
    assert stats.kstest(2 * Y[:: 4 * H], stats.chi2(H * (H + 1)).cdf).pvalue > 1e-3


def library_route(spec, zmax, B, C, thr, numharm):
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
    out = []
    for H in range(1, numharm + 1):
        Y = reshape_route(P, H)
        nH = Y.size
        pre = np.concatenate([[0.0], np.cumsum(Y)])
        for c in range((nH + C - 1) // C):
            lo, hi = c * C, min((c + 1) * C, nH)
            best = None
            for w in range(1, zmax + 1):
                i = np.arange(lo, min(hi, nH - w + 1))
                if i.size == 0:
                    continue
                S = pre[i + w] - pre[i]
                k = int(np.argmax(S))
                lnp = min(0.0, stats.chi2.logsf(2 * S[k], H * (H + 1) * w))          # L220: k = H(H+1)(z+1)
                if best is None or lnp < best[0]:
                    best = (lnp, int(i[k]), w, S[k])
            if best is not None and best[0] <= special.log_ndtr(-thr):
                out.append((H, best[1], best[2], best[3], stats.norm.isf(np.exp(best[0]))))
    return out


@pytest.mark.parametrize("seed,n,zmax,B,C,thr,numharm", [(0, 513, 8, 128, 16, 2.5, 4), (1, 1025, 12, 256, 40, 3.0, 3),
                                                          (2, 300, 6, 512, 7, 2.0, 2)])
def test_search_harmonics_matches_library_route(orc, seed, n, zmax, B, C, thr, numharm):
    rng = np.random.default_rng(seed)
    spec = (rng.normal(0, 30, n) + 1j * rng.normal(0, 30, n)).astype(np.complex64)
    for h in range(1, 5):
        spec[h * 23: h * 23 + 2] *= 3.0                                  # power at 23 and its harmonics
    got = orc.search_harmonics(spec, zmax, B, C, thr, numharm)
    ref = library_route(spec, zmax, B, C, thr, numharm)
    assert len(got) == len(ref) > 0
    for g, r in zip(got, ref):
        assert (g["numharm"], g["bin"], g["width"]) == (r[0], r[1], r[2])
        assert g["power"] == pytest.approx(r[3], rel=1e-11)
        assert g["sigma"] == pytest.approx(r[4], abs=1e-7)
    plain = orc.search(spec, zmax, B, C, thr)
    h1 = got[got["numharm"] == 1]
    assert np.array_equal(h1, plain)                                     # numharm = 1 is the plain search


def test_harmonics_add_up(orc):
    # a narrow pulse train puts similar power into the fundamental and its harmonics (L203): summing 4 of them must beat
    # the fundamental alone at the fundamental's bin
    n, r0 = 8193, 301
    rng = np.random.default_rng(9)
    spec = (rng.normal(0, 10, n) + 1j * rng.normal(0, 10, n)).astype(np.complex64)
    for h in range(1, 5):
        spec[h * r0] += 45.0
    got = orc.search_harmonics(spec, 4, 1024, 50, 3.0, 4)
    best = {H: got[(got["numharm"] == H) & (np.abs(got["bin"] - r0) <= 1)]["sigma"].max() for H in (1, 4)}
    assert best[4] > best[1] + 1.5


def test_per_width_emission_with_harmonics_matches_library_route(orc):
    """orc_search_opts(per_width = 1) at numharm 3: every (H, block, width) whose maximum passes chi2.logsf(2S, H(H+1)w) (L220;
    Alg. 4), through numpy/scipy only; and the default output is the highest-sigma record of each (H, block)."""
    n, zmax, B, C, thr, numharm = 1025, 9, 256, 40, 2.5, 3
    rng = np.random.default_rng(31)
    spec = (rng.normal(0, 30, n) + 1j * rng.normal(0, 30, n)).astype(np.complex64)
    for h in range(1, 4):
        spec[h * 41: h * 41 + 2] *= 3.0
    got = orc.search_harmonics(spec, zmax, B, C, thr, numharm, per_width=True)
    P = orc.normalise_power(spec, B)        # pinned on its own (tests/test_oracle_normalise.py)
    want = []
    for H in range(1, numharm + 1):
        Y = reshape_route(P, H)
        nH = Y.size
        pre = np.concatenate([[0.0], np.cumsum(Y)])
        for c in range((nH + C - 1) // C):
            lo, hi = c * C, min((c + 1) * C, nH)
            for w in range(1, zmax + 1):
                i = np.arange(lo, min(hi, nH - w + 1))
                if i.size == 0:
                    continue
                S = pre[i + w] - pre[i]
                k = int(np.argmax(S))
                if stats.chi2.logsf(2 * S[k], H * (H + 1) * w) <= special.log_ndtr(-thr):
                    want.append((H, int(i[k]), w, S[k]))
    assert [(int(g["numharm"]), int(g["bin"]), int(g["width"])) for g in got] == [w[:3] for w in want]
    assert len({w[0] for w in want}) == numharm and len(want) > 30
    assert np.allclose(got["power"], [w[3] for w in want], rtol=1e-11)
    best = orc.search_harmonics(spec, zmax, B, C, thr, numharm)
    for r in best:
        mine = got[(got["numharm"] == r["numharm"]) & (got["bin"] // C == r["bin"] // C)]
        top = mine[np.argmax(mine["sigma"])]
        assert (top["bin"], top["width"], top["sigma"]) == (r["bin"], r["width"], r["sigma"])
