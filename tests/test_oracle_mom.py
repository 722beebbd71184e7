"""Pins for the oracle's Algorithm 1 (the paper's approximate GPU normalisation)."""
import numpy as np
import pytest
from scipy import stats


def numpy_route(v):
    """Alg. 1's strided grouping through numpy.median (the median of 4 = (a+b+c+d−min−max)/2)."""
    v = np.asarray(v, dtype=np.float64)
    while v.size >= 4:
        v = np.median(v.reshape(4, v.size // 4), axis=0)      # element i of row j is sdata[i + j·stride]
    return float(v.mean())


@pytest.mark.parametrize("n", [4, 16, 64, 1024, 4096, 2, 8, 32, 2048, 8192])
def test_median_of_medians_matches_numpy_route(orc, n):
    rng = np.random.default_rng(n)
    v = rng.normal(3.0, 10.0, n)
    assert orc.median_of_medians(v) == pytest.approx(numpy_route(v), rel=1e-14, abs=1e-14)
    if n == 4:
        assert orc.median_of_medians(v) == pytest.approx(np.median(v), rel=1e-15)
    if n == 2:
        assert orc.median_of_medians(v) == pytest.approx(v.mean(), rel=1e-15)


def test_median_of_medians_hand_example(orc):
    # 16 values, strides 4 then 1: groups are the columns of the 4 x 4 row-major table (L636-642)
    v = [1, 9, 2, 8,
         7, 3, 6, 4,
         5, 5, 9, 0,
         2, 6, 1, 7]
    # columns: (1,7,5,2)->3.5  (9,3,5,6)->5.5  (2,6,9,1)->4  (8,4,0,7)->5.5 ; then (3.5,5.5,4,5.5) -> 4.75
    assert orc.median_of_medians(v) == 4.75


def test_median_of_medians_is_an_estimate_of_the_median(orc):
    rng = np.random.default_rng(7)
    err = [orc.median_of_medians(rng.normal(0, 1, 4096)) for _ in range(200)]
    assert abs(np.mean(err)) < 0.02 and 0.01 < np.std(err) < 0.06        # unbiased, a few % of sigma (exact: 0.0196)


def test_normalise_power_mom_statistics_and_tail(orc):
    rng = np.random.default_rng(3)
    n, B = 4 * 1024 + 5, 1024
    spec = (rng.normal(2.0, 30, n) + 1j * rng.normal(-1.0, 30, n)).astype(np.complex64)
    P = orc.normalise_power_mom(spec, B)
    exact = orc.normalise_power(spec, B)
    # Alg. 1 is biased: the median of 4 averages the two middle values, which over-estimates the median of the skewed
    # |deviation| distribution by ≈ 6 %, so powers come out ≈ 12 % low (0.88 instead of 1) — exponential all the same (L150)
    assert P.mean() == pytest.approx(0.88, abs=0.05) and stats.kstest(P / P.mean(), "expon").pvalue > 1e-4
    ratio = P / exact
    assert 0.8 < np.median(ratio) < 0.95 and np.std(ratio) < 0.15            # a per-block scale error, not noise
    # the 5 bins after the last chunk use the last chunk's median and MAD (R30): recompute them through the numpy route
    lo = 3 * B
    m = [numpy_route(part[lo:lo + B].astype(np.float64)) for part in (spec.real, spec.imag)]
    s = [1.4826 * numpy_route(np.abs(part[lo:lo + B].astype(np.float64) - mm)) for part, mm in zip((spec.real, spec.imag), m)]
    k = n - 1
    want = 0.5 * (((float(spec.real[k]) - m[0]) / s[0]) ** 2 + ((float(spec.imag[k]) - m[1]) / s[1]) ** 2)
    assert P[k] == pytest.approx(want, rel=1e-12)


def test_search_with_mom_differs_only_through_the_normalisation(orc):
    rng = np.random.default_rng(5)
    n = 4096 + 1
    spec = (rng.normal(0, 30, n) + 1j * rng.normal(0, 30, n)).astype(np.complex64)
    spec[1000:1008] *= 3.0
    a = orc.search_harmonics(spec, 16, 1024, 64, 3.0, 1, median_of_medians=True)
    b = orc.search(spec, 16, 1024, 64, 3.0)
    assert 0 < len(a) <= len(b)                               # powers ≈ 12 % low: the marginal candidates drop out
    top_a, top_b = a[np.argmax(a["sigma"])], b[np.argmax(b["sigma"])]
    assert abs(int(top_a["bin"]) - int(top_b["bin"])) <= 2 and 0.0 < top_b["sigma"] - top_a["sigma"] < 1.5


def mom_power_numpy_route(spec, B):
    """orc_normalise_power_mom through the numpy route: every bin of every chunk, the tail after the last chunk included (R30)."""
    n = spec.size
    nb = n // B
    P = np.empty(n)
    for j in range(nb):
        lo, hi = j * B, (n if j == nb - 1 else (j + 1) * B)
        comps = []
        for part in (spec.real, spec.imag):
            chunk = part[lo:lo + B].astype(np.float64)
            m = numpy_route(chunk)
            s = 1.4826 * numpy_route(np.abs(chunk - m))
            comps.append((part[lo:hi].astype(np.float64) - m) / s)
        P[lo:hi] = 0.5 * (comps[0] ** 2 + comps[1] ** 2)
    return P


@pytest.mark.parametrize("n,B", [(4 * 1024 + 5, 1024), (3 * 256, 256), (2 * 2048 + 1000, 2048), (8192 + 1, 8192), (5 * 512 + 511, 512)])
def test_normalise_power_mom_matches_numpy_route_on_every_bin(orc, n, B):
    rng = np.random.default_rng(n + B)
    spec = (rng.normal(2.0, 30, n) + 1j * rng.normal(-1.0, 7, n)).astype(np.complex64)
    P = orc.normalise_power_mom(spec, B)
    want = mom_power_numpy_route(spec, B)
    assert np.allclose(P, want, rtol=1e-11, atol=0.0)


def test_search_with_mom_matches_library_route(orc):
    """orc_search_opts(norm_mode = 1): Alg. 1 powers through the numpy route, then cumsum differences, chi2.logsf, norm.isf."""
    from scipy import special
    n, zmax, B, C, thr = 1024 + 300, 10, 256, 48, 2.5
    rng = np.random.default_rng(77)
    spec = (rng.normal(0, 30, n) + 1j * rng.normal(0, 30, n)).astype(np.complex64)
    spec[400:405] *= 3.5
    got = orc.search_harmonics(spec, zmax, B, C, thr, 1, median_of_medians=True)
    P = mom_power_numpy_route(spec, B)
    pre = np.concatenate([[0.0], np.cumsum(P)])
    ref = []
    for c in range((n + C - 1) // C):
        lo, hi = c * C, min((c + 1) * C, n)
        best = None
        for w in range(1, zmax + 1):
            i = np.arange(lo, min(hi, n - w + 1))
            if i.size == 0:
                continue
            S = pre[i + w] - pre[i]
            k = int(np.argmax(S))
            lnp = min(0.0, stats.chi2.logsf(2 * S[k], 2 * w))
            if best is None or lnp < best[0]:
                best = (lnp, int(i[k]), w, S[k])
        if best is not None and best[0] <= special.log_ndtr(-thr):
            ref.append(best)
    assert len(got) == len(ref) > 0
    for g, r in zip(got, ref):
        assert (g["bin"], g["width"]) == (r[1], r[2])
        assert g["power"] == pytest.approx(r[3], rel=1e-10)
        assert g["sigma"] == pytest.approx(stats.norm.isf(np.exp(r[0])), abs=1e-7)
