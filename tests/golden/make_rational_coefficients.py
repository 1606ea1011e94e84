"""Writes tests/golden/rational_coefficients.txt from oracle/rational.py ONLY (50-digit mpmath): the
eq. 8 coefficients of the minimax approximations the paper uses, b = -2 and b = 4
(PAPER.md:131), for a few (n, xmin, xmax).  Never run against the CUDA library.

    python tests/golden/make_rational_coefficients.py
"""
import os
import sys
from fractions import Fraction

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

from oracle import rational as R  # noqa: E402

CASES = [(-1, 2, 6, 1e-3, 8.5), (-1, 2, 12, 1.25e-5, 8.5), (1, 4, 6, 1e-3, 8.5), (1, 4, 12, 1.25e-5, 8.5)]
OUT = os.path.join(os.path.dirname(os.path.abspath(__file__)), "rational_coefficients.txt")


def main():
    with open(OUT, "w") as fh:
        fh.write("# Minimax (relative error) approximations x^(num/den) ~= c0 + sum_k c_k/(x + d_k) on [xmin, xmax]\n"
                 "# (eq. 8, PAPER.md:133; b = -2 and b = 4 of PAPER.md:131), produced by\n"
                 "# tests/golden/make_rational_coefficients.py from oracle/rational.py (mpmath, 50 digits):\n"
                 "# num/den = -1/2 by Zolotarev's closed form, 1/4 by the Remez exchange.  The paper prints no\n"
                 "# coefficients; these rows are the oracle's, pinned by tests/test_oracle_rational.py.\n"
                 "# case num den n xmin xmax delta c0\n#   k c_k d_k\n")
        for num, den, n, lo, hi in CASES:
            z = (R.zolotarev_inv_sqrt(n, lo, hi) if (num, den) == (-1, 2)
                 else R.minimax_pow(Fraction(num, den), n, lo, hi))
            fh.write(f"case {num} {den} {n} {lo!r} {hi!r} {z['delta']!r} {z['c0']!r}\n")
            for k in range(n):
                fh.write(f"  {k} {float(z['c'][k])!r} {float(z['d'][k])!r}\n")


if __name__ == "__main__":
    main()
