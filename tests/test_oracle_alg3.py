"""Pins for the oracle's Algorithm 3 (§2.6 Eq. 10-12): the paper's polynomial ln p.

It is an approximation obtained by regression, so there is no closed form to meet: the pins are the numbers the listing prints
(f(0) = −755.24091, A_1 = 1500, the `dof >= pow × 1.05` branch), an exact rational evaluation of the printed polynomial
(fractions.Fraction on the decimal strings, typed here independently of the C source), the χ² tail's slope it must approach
(ln p → −pow/2), and its measured error against the exact tail (orc_ln_q, itself pinned to mpmath) where it is usable."""
from fractions import Fraction

import numpy as np
import pytest

# the listing's coefficients, highest power first (x^16 … x^0), as printed at PAPER.md:L661
PRINTED = ["-4.4604059e-46", "9.4927863e-42", "-9.1470451e-38", "5.2810851e-34", "-2.0376166e-30", "5.5480334e-27",
           "-1.0973877e-23", "1.5991804e-20", "-1.7231488e-17", "1.3660070e-14", "-7.8617952e-12", "3.2136336e-9",
           "-9.0466418e-7", "0.00016945948", "-0.021494231", "2.9515954", "-755.24091"]


def exact_logp(power: Fraction, dof: Fraction) -> Fraction:
    x = 1500 * dof / power
    f = Fraction(0)
    for k, c in enumerate(PRINTED):
        f += Fraction(c) * x ** (16 - k)
    return power * f / 1500


def test_printed_constants(orc):
    assert len(PRINTED) == 17
    # x = 0 (no degrees of freedom): only the constant term is left, logp = pow × (−755.24091)/1500
    for p in (1.0, 41.4, 3000.0):
        assert orc.power_to_logp(p, 0.0) == pytest.approx(p * -755.24091 / 1500.0, rel=1e-15)
    # the branch of the listing: dof >= pow × 1.05 → 0.0 exactly
    assert orc.power_to_logp(100.0, 105.0) == 0.0 and orc.power_to_logp(100.0, 300.0) == 0.0
    assert orc.power_to_logp(100.0, 104.99) != 0.0


@pytest.mark.parametrize("power,dof", [("41.4", "2"), ("60", "2"), ("108", "26"), ("300", "128"), ("600", "400"), ("782", "400"),
                                        ("250", "200"), ("1000", "64"), ("3000", "2400"), ("2500", "2600")])
def test_matches_exact_rational_evaluation_of_the_printed_polynomial(orc, power, dof):
    want = float(exact_logp(Fraction(power), Fraction(dof)))
    got = orc.power_to_logp(float(power), float(dof))
    x = 1500.0 * float(dof) / float(power)
    # in double the terms (up to ~1e9 in magnitude at x ≈ 1400) cancel: absolute error ≲ 1e-16 × Σ|term| × pow/1500
    terms = sum(abs(float(c)) * x ** (16 - k) for k, c in enumerate(PRINTED))
    assert got == pytest.approx(want, abs=4e-16 * terms * float(power) / 1500.0 + 1e-12)
    # a dropped term, a wrong sign or a transposed exponent changes the value by far more than that
    for k in (0, 5, 12, 15):
        broken = want - 2 * float(Fraction(PRINTED[k])) * x ** (16 - k) * float(power) / 1500.0
        assert abs(broken - got) > 1e3 * (4e-16 * terms * float(power) / 1500.0 + 1e-12) or x < 600


def test_tail_slope_is_minus_half(orc):
    # far in the tail (pow >> dof) the χ² survival function falls like e^{−pow/2}: Alg. 3's constant term gives −0.5035
    for dof in (2.0, 20.0):
        assert orc.power_to_logp(1e5, dof) / 1e5 == pytest.approx(-0.5, abs=5e-3)


def test_error_against_the_exact_tail(orc):
    """Where Alg. 3 is usable (x = 1500·dof/pow ≲ 1000) it is LESS significant than the exact tail by 0 … 5 nats; beyond
    x ≈ 1100 the printed 8-digit coefficients no longer determine f (terms ~1e8-1e9 cancel) and it diverges: at dof 2400,
    pow 3000 it gives −69.5 against the exact −35.3."""
    worst = 0.0
    for w in (1, 2, 4, 8, 13, 32, 64, 100, 128):
        T = orc.power_threshold(w, 6.0)
        for S in np.linspace(T, 3.0 * T, 25):
            if 1500.0 * w / S > 1000.0:
                continue
            d = orc.power_to_logp(2.0 * S, 2.0 * w) - orc.ln_q(w, S)
            assert -0.25 <= d <= 5.0, (w, S, d)
            worst = max(worst, d)
    assert 3.0 < worst <= 5.0
    assert orc.power_to_logp(3000.0, 2400.0) == pytest.approx(-69.5, abs=0.1) and orc.ln_q(1200, 1500.0) == pytest.approx(-35.32, abs=0.01)


def test_search_with_alg3_matches_numpy_route(orc):
    """orc_search_all(signif_mode = 1): the plumbing (units pow = 2S, dof = H(H+1)·w; reduction over widths; threshold) through
    numpy.polyval on the printed coefficients over the oracle's own (separately pinned) block maxima."""
    from scipy import special, stats
    n, zmax, B, C, thr, numharm = 1025, 12, 256, 40, 3.0, 2
    rng = np.random.default_rng(91)
    spec = (rng.normal(0, 30, n) + 1j * rng.normal(0, 30, n)).astype(np.complex64)
    spec[300:304] *= 4.0
    spec[600:602] *= 5.0
    got = orc.search_harmonics(spec, zmax, B, C, thr, numharm, poly_logp=True)
    coef = [float(c) for c in PRINTED]
    P = orc.normalise_power(spec, B)
    want = []
    for H in range(1, numharm + 1):
        Y = orc.harmonic_sum(P, H)
        M, I = orc.block_maxima(Y, zmax, C)
        for c in range(M.shape[0]):
            best = None
            for w in range(1, zmax + 1):
                if I[c, w - 1] < 0:
                    continue
                powr, dof = 2.0 * M[c, w - 1], float(H * (H + 1) * w)
                lnp = 0.0 if dof >= 1.05 * powr else powr * np.polyval(coef, 1500.0 * dof / powr) / 1500.0
                lnp = min(0.0, lnp)
                if best is None or lnp < best[0]:
                    best = (lnp, int(I[c, w - 1]), w, M[c, w - 1])
            if best is not None and best[0] <= special.log_ndtr(-thr):
                want.append((H, best[1], best[2], best[3], stats.norm.isf(np.exp(best[0]))))
    assert len(got) == len(want) > 3
    for g, r in zip(got, want):
        assert (g["numharm"], g["bin"], g["width"]) == r[:3]
        assert g["power"] == pytest.approx(r[3], rel=1e-12) and g["sigma"] == pytest.approx(r[4], abs=1e-7)
    exact = orc.search_harmonics(spec, zmax, B, C, thr, numharm)
    assert len(got) <= len(exact)          # Alg. 3 under-states the significance of narrow widths: marginal candidates drop out
