"""Pins for the oracle's significance (Eq. 9; L114): mpmath table, scipy routines, closed forms."""
from pathlib import Path

import numpy as np
import pytest
from scipy import special, stats

PINS = [ln.split() for ln in (Path(__file__).parent / "golden" / "significance_pins.txt").read_text().splitlines()
        if ln and not ln.startswith("#")]


@pytest.mark.parametrize("w,S,lnp,sigma", PINS)
def test_mpmath_pins(orc, w, S, lnp, sigma):
    w, S, lnp, sigma = int(w), float(S), float(lnp), float(sigma)
    got = orc.ln_q(w, S)
    # abs: ln Q near 0 is a difference of O(100) terms; for the harmonic search's large shapes ln Q is what is left of
    # three terms of size w·ln w ≈ 4e5 (−S + k·ln S − lnΓ(k+1)), each carrying a relative 1e-16
    assert got == pytest.approx(lnp, rel=2e-12, abs=1e-12 if w <= 1200 else 2e-9)
    assert orc.sigma_from_lnp(lnp) == pytest.approx(sigma, abs=2e-9)
    if w > 1200 and lnp < -1.0:     # a mistake of one term, or of one unit of shape, moves ln p by far more than this
        assert abs(orc.ln_q(w - 1, S) - got) > 1e-3 and abs(orc.ln_q(w + 1, S) - got) > 1e-3


def test_width_one_is_exponential_tail(orc):
    for S in (0.1, 1.0, 20.7, 500.0):
        assert orc.ln_q(1, S) == pytest.approx(-S, rel=1e-15)


@pytest.mark.parametrize("w", [1, 2, 3, 7, 32, 200, 1200, 2000, 12000, 40960])
def test_against_scipy_gammaincc_and_chi2(orc, w):
    hi = 1.6 * w + 30 if w <= 1200 else w + 12 * np.sqrt(w)      # beyond ≈ 12 sd gammaincc underflows for the large shapes
    for S in np.linspace(0.3 * w, hi, 9):
        ref = np.log(special.gammaincc(w, S))
        if np.isfinite(ref):
            assert orc.ln_q(w, S) == pytest.approx(ref, rel=1e-10, abs=1e-12 if w <= 1200 else 1e-8)
        assert orc.ln_q(w, S) == pytest.approx(stats.chi2.logsf(2 * S, 2 * w), rel=1e-9, abs=1e-12 if w <= 1200 else 1e-8)


def test_closed_form_finite_sum(orc):
    from math import exp, factorial, log
    for w, S in [(2, 3.0), (4, 9.5), (6, 1.25)]:
        q = exp(-S) * sum(S ** k / factorial(k) for k in range(w))
        assert orc.ln_q(w, S) == pytest.approx(log(q), rel=1e-13)


def test_monotone(orc):
    for w in (1, 5, 64, 700):
        vals = np.array([orc.ln_q(w, S) for S in np.linspace(0.5, 3 * w + 50, 200)])
        assert np.all(np.diff(vals) < 1e-12)          # more power → smaller p (rounding noise only where p ≈ 1)
        tail = vals < -1e-6
        assert np.all(np.diff(vals[tail]) < 0)
    for S in (10.0, 200.0):
        vals = np.array([orc.ln_q(w, S) for w in range(1, 300)])
        assert np.all(np.diff(vals) > -1e-12)         # same power over more bins → larger p
        tail = vals < -1e-6
        assert np.all(np.diff(vals[tail]) > 0)


def test_ln_sf_and_sigma_against_scipy(orc):
    for x in (-8.0, -1.0, 0.0, 0.5, 3.0, 6.0, 7.0, 15.0, 29.9, 30.0, 30.1, 37.0, 60.0, 400.0):
        assert orc.ln_sf(x) == pytest.approx(special.log_ndtr(-x), rel=1e-12, abs=1e-16)
    for p in (0.4, 1e-3, 1e-9, 1e-30, 1e-300):
        assert orc.sigma_from_lnp(np.log(p)) == pytest.approx(stats.norm.isf(p), abs=1e-9)
    # R17 constants: ln sf(6), ln sf(7)
    assert orc.ln_sf(6.0) == pytest.approx(-20.7367689499747, abs=1e-10)
    assert orc.ln_sf(7.0) == pytest.approx(-27.3843074988111, abs=1e-10)


def test_power_thresholds_round_trip(orc):
    # T_w with σ(T_w, w) = threshold: values derived in SURVEY.md §8(c) (single-trial σ = 6 / 7)
    table = {1: (20.7368, 27.3843), 2: (23.9538, 30.8452), 13: (47.3151, 55.9198), 100: (172.1023, 186.7300),
             200: (296.8369, 315.5281), 1200: (1419.6481, 1458.7153)}
    for w, (t6, t7) in table.items():
        assert orc.power_threshold(w, 6.0) == pytest.approx(t6, abs=2e-4)
        assert orc.power_threshold(w, 7.0) == pytest.approx(t7, abs=2e-4)
        assert orc.sigma_from_lnp(orc.ln_q(w, orc.power_threshold(w, 6.0))) == pytest.approx(6.0, abs=1e-9)
    # Bonferroni: N trials shift ln p by ln N (R15)
    assert orc.ln_q(5, orc.power_threshold(5, 6.0, n_trials=1e6)) == pytest.approx(orc.ln_sf(6.0) - np.log(1e6), abs=1e-9)
