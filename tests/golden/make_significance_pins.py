"""Writes significance_pins.txt: 50-digit reference values of the χ² tail and its Gaussian-equivalent σ.

Independent of both the oracle and the CUDA path: uses only mpmath.  The quantities are those of
PAPER.md:L154-158 (Eq. 9: a width-w boxcar of normalised powers is χ² with 2w degrees of freedom; p = survival
function; p → Gaussian-equivalent σ through the normal survival function, L114/L158), in mean-1 power units
(χ² statistic = 2S):

    ln p  = ln Q(w, S),  Q = regularised upper incomplete gamma  (= chi2.sf(2S, 2w))
    sigma = x with ½ erfc(x/√2) = p

Run:  python tests/golden/make_significance_pins.py
"""
from pathlib import Path

import mpmath as mp

mp.mp.dps = 50

CASES = [
    (1, "10"), (1, "20.72326583694641"), (1, "50"), (2, "24.2"), (3, "26.7"), (4, "30"), (8, "37.8435"), (13, "54"),
    (16, "52.6057"), (32, "80"), (64, "128"), (100, "180"), (128, "207.9386"), (200, "300"), (200, "391"),
    (256, "363.9496"), (512, "659.6351"), (1024, "1227.8128"), (1200, "1419.6481"), (1200, "1500"), (1200, "1600"),
    (1200, "3000"), (5, "5"), (10, "10"), (50, "30"), (200, "150"), (7, "0.5"), (1, "700"), (3, "1000"),
    # Gamma shapes the harmonic search reaches (w·H(H+1)/2: 2000 at zmax 200 / numharm 4, 12000 at zmax 1200, 40960 at
    # PULSCAN_MAX_ZMAX): a power just above the σ = 6 threshold, a strong one, and one below the mean (largest term inside the sum)
    (2000, "2281"), (2000, "2600"), (2000, "1950"), (12000, "12672"), (12000, "13500"), (12000, "11900"),
    (40960, "42190"), (40960, "44000"), (40960, "40800"),
]


def ln_q(w, S):
    return mp.log(mp.gammainc(w, S, mp.inf, regularized=True))


def sigma(lnp):
    p_target = lnp
    f = lambda x: mp.log(mp.erfc(x / mp.sqrt(2)) / 2) - p_target
    x0 = mp.sqrt(max(mp.mpf(1), -2 * lnp))
    return mp.findroot(f, x0, tol=mp.mpf(10) ** -40)


def main():
    lines = ["# w  S  ln_p  sigma   (mpmath, 50 digits; PAPER.md Eq. 9 L156, L114, L158; mean-1 units)"]
    for w, s in CASES:
        S = mp.mpf(s)
        lp = ln_q(w, S)
        sg = sigma(lp)
        lines.append(f"{w} {s} {mp.nstr(lp, 20)} {mp.nstr(sg, 20)}")
    Path(__file__).with_name("significance_pins.txt").write_text("\n".join(lines) + "\n")


if __name__ == "__main__":
    main()
