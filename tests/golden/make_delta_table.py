"""Writes tests/golden/delta_table.txt: delta(n, eps) = max_{eps<=y<=1} |1 - sqrt(y) P_n(y)| of eq. 2.6 for the
Chebyshev-interpolation coefficients (R7) and for the min-max coefficients (R18), computed by the ORACLE alone
(oracle/sign.py).  PAPER.md prints no worked values of its own (its tables hold timings on a GTX 285 only), so this is the
one stored fixture: a regression anchor for both coefficient routines and for the library's host utilities, which are compared
with it in tests/test_golden.py.

    python tests/golden/make_delta_table.py
"""
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

from oracle import sign as osign  # noqa: E402

CASES = [(20, 0.05), (40, 0.02), (60, 0.01), (100, 0.01), (100, 0.005), (100, 0.002), (200, 0.002), (200, 0.001)]
MINMAX = [(20, 0.05), (40, 0.02), (60, 0.01)]


def main():
    lines = ["# n eps kind delta   (written by tests/golden/make_delta_table.py from oracle/sign.py; eq. 2.6, PAPER.md:L68-73)"]
    for n, eps in CASES:
        c = osign.cheb_coeffs(n, eps)
        lines.append(f"{n} {eps} interpolation {osign.measure_delta(c, eps):.6e}")
    for n, eps in MINMAX:
        c, delta, levelled = osign.minmax_coeffs(n, eps)
        lines.append(f"{n} {eps} minmax {delta:.6e}")
    with open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "delta_table.txt"), "w") as f:
        f.write("\n".join(lines) + "\n")


if __name__ == "__main__":
    main()
