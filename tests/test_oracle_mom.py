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
