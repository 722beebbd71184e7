"""Pins for the oracle's normalisation + power (Eq. 8): library routines, invariants, statistics."""
import numpy as np
import pytest
from scipy import stats


def test_kappa_is_inverse_normal_quantile(orc):
    # PAPER.md:L142 "scaled by the factor 1/φ⁻¹(3/4)"; Alg. 1 L648 prints 1.4826
    assert orc.kappa() == pytest.approx(1.0 / stats.norm.ppf(0.75), rel=1e-15)
    assert round(orc.kappa(), 4) == 1.4826


@pytest.mark.parametrize("n", [1, 2, 3, 4, 7, 8, 255, 256, 1025])
def test_median_matches_numpy(orc, n):
    rng = np.random.default_rng(n)
    v = rng.normal(size=n)
    assert orc.median(v) == np.median(v)
    v[: n // 2] = v[0]  # duplicates
    assert orc.median(v) == np.median(v)


def test_median_even_is_mean_of_central_pair(orc):
    # Alg. 1 local_median(a,b,c,d) = (a+b+c+d-min-max)/2
    a = np.array([4.0, 1.0, 3.0, 10.0])
    assert orc.median(a) == (a.sum() - a.min() - a.max()) / 2 == 3.5


@pytest.mark.parametrize("n", [5, 64, 1001, 4096])
def test_normalise_block_matches_scipy_mad(orc, n):
    rng = np.random.default_rng(100 + n)
    v = rng.normal(3.0, 17.0, size=n)
    out, med, scale = orc.normalise_block(v)
    mad_n = stats.median_abs_deviation(v, scale="normal")  # = MAD / Φ⁻¹(3/4)
    assert med == np.median(v)
    assert scale == pytest.approx(mad_n, rel=1e-14)
    np.testing.assert_allclose(out, (v - np.median(v)) / mad_n, rtol=1e-13, atol=0)


def test_normalised_block_has_median0_and_unit_scaled_mad(orc):
    rng = np.random.default_rng(5)
    v = rng.normal(-2.0, 0.01, size=2049)
    out, _, _ = orc.normalise_block(v)
    assert abs(np.median(out)) < 1e-15
    assert stats.median_abs_deviation(out, scale="normal") == pytest.approx(1.0, rel=1e-13)


def test_scale_and_offset_invariance(orc):
    rng = np.random.default_rng(6)
    v = rng.normal(size=512).astype(np.float32).astype(np.float64)
    a, _, _ = orc.normalise_block(v)
    b, _, _ = orc.normalise_block(v * 2.0 ** 7)   # power-of-two scaling is exact → bit-identical
    assert np.array_equal(a, b)
    c, _, _ = orc.normalise_block(v + 1024.0)     # exact for float32-valued inputs of this size
    np.testing.assert_allclose(a, c, rtol=0, atol=1e-9)


def test_zero_mad_gives_zero_block(orc):
    v = np.full(33, 2.5)
    v[3] = 9.0
    out, med, scale = orc.normalise_block(v)
    assert med == 2.5 and scale == 0.0 and np.all(out == 0.0)


def _numpy_normalise_power(spec, B):
    """Independent route: numpy.median + scipy MAD per block, last block absorbs the remainder (R6)."""
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
    return P


@pytest.mark.parametrize("n,B", [(64, 16), (65, 16), (79, 16), (1025, 256), (10, 16), (4097, 1024)])
def test_normalise_power_blocks_and_remainder(orc, n, B):
    rng = np.random.default_rng(n * 31 + B)
    spec = (rng.normal(0, 50, n) + 1j * rng.normal(2, 70, n)).astype(np.complex64)
    P = orc.normalise_power(spec, B)
    np.testing.assert_allclose(P, _numpy_normalise_power(spec, B), rtol=1e-12, atol=1e-300)


def test_components_are_normalised_independently(orc):
    # "Each component, real and imaginary ... normalised independently"
    rng = np.random.default_rng(9)
    n, B = 512, 128
    re, im = rng.normal(0, 3, n), rng.normal(0, 3, n)
    P1 = orc.normalise_power((re + 1j * im).astype(np.complex64), B)
    P2 = orc.normalise_power((re + 1j * (1000 * im + 5)).astype(np.complex64), B)  # affine change of im only
    np.testing.assert_allclose(P1, P2, rtol=1e-5)


def test_white_noise_power_is_exponential_mean_one(orc):
    # |X'|² ~ χ²(2) per bin; in mean-1 units (R2) P ~ Exp(1)
    rng = np.random.default_rng(11)
    n = 1 << 17
    spec = (rng.normal(0, 181.0, n) + 1j * rng.normal(0, 181.0, n)).astype(np.complex64)
    P = orc.normalise_power(spec, 4096)
    assert P.mean() == pytest.approx(1.0, abs=0.02)
    assert stats.kstest(P[::7], "expon").pvalue > 1e-3
    for t in (1.0, 3.0, 6.0):
        assert (P > t).mean() == pytest.approx(np.exp(-t), rel=0.15)
