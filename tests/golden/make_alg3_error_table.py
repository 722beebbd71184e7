"""Writes alg3_error_table.txt: the error profile of the paper's polynomial ln p (Alg. 3) against the exact
chi-squared tail, over (Gamma shape = d.o.f./2, significance of the exact value).  Calls only oracle/ (orc_power_to_logp,
orc_ln_q, orc_power_threshold, orc_sigma_from_lnp — each pinned in tests/test_oracle_*.py).  DESIGN.md §9 quotes this table.

Run:  python tests/golden/make_alg3_error_table.py
"""
import sys
from pathlib import Path

ROOT = Path(__file__).resolve().parents[2]
sys.path.insert(0, str(ROOT))
import oracle  # noqa: E402

SHAPES = [1, 2, 4, 8, 16, 32, 64, 100, 128, 150, 200, 256, 400, 600, 1200, 2000]
SIGMAS = [6.0, 8.0, 12.0, 20.0, 40.0]


def main():
    oracle.build()
    lines = ["# shape  sigma_exact  S  x=1500*dof/pow  lnp_exact  lnp_alg3  diff   (mean-1 units: pow = 2S, dof = 2*shape; R31)"]
    for k in SHAPES:
        for sg in SIGMAS:
            S = oracle.power_threshold(k, sg)
            exact = oracle.ln_q(k, S)
            poly = oracle.power_to_logp(2.0 * S, 2.0 * k)
            lines.append(f"{k} {sg:g} {S:.6f} {1500.0 * k / S:.2f} {exact:.6f} {poly:.6f} {poly - exact:+.4f}")
    Path(__file__).with_name("alg3_error_table.txt").write_text("\n".join(lines) + "\n")


if __name__ == "__main__":
    main()
