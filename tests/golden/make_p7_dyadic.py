"""Writes tests/golden/p7_dyadic.txt: the exact SNR of a 3-filter template on an 8-sample input.

Independent of both oracle/ and the CUDA path: the defining recurrence (BASELINE.json:north_star;
SURVEY.md §8(c) pin P7) is evaluated in exact rational arithmetic (fractions.Fraction).  All
coefficients and inputs are dyadic rationals, so every intermediate is exactly representable in
float32 and float64 and both the oracle and the GPU must reproduce these values BITWISE.
The first four entries were also re-derived by hand.
"""
from fractions import Fraction as F
from pathlib import Path

FILTERS = [  # (a1_re, a1_im, b0_re, b0_im, delay)
    (F(1, 2), F(0), F(1), F(0), 0),
    (F(0), F(1, 2), F(1), F(1), 1),
    (F(1, 2), F(-1, 2), F(0), F(-1, 2), 3),
]
X = [1, 2, 0, -1, 0, 0, 4, 0]


def exact_snr():
    y = [(F(0), F(0)) for _ in FILTERS]
    out = []
    for n in range(len(X)):
        sre, sim = F(0), F(0)
        for k, (are, aim, bre, bim, d) in enumerate(FILTERS):
            xd = F(X[n - d]) if n - d >= 0 else F(0)
            yre, yim = y[k]
            y[k] = (are * yre - aim * yim + bre * xd, are * yim + aim * yre + bim * xd)
            sre += y[k][0]
            sim += y[k][1]
        out.append((sre, sim))
    return out


if __name__ == "__main__":
    lines = ["# P7 exact golden vector (SURVEY.md §8(c)); definition: BASELINE.json:north_star recurrence.",
             "# Written by tests/golden/make_p7_dyadic.py with exact rational arithmetic (no oracle, no GPU).",
             "# filters (a1_re a1_im b0_re b0_im delay):"]
    lines += ["# " + " ".join(str(v) for v in f) for f in FILTERS]
    lines += ["# x: " + " ".join(str(v) for v in X), "# n  SNR_re  SNR_im   (exact fractions)"]
    for n, (re, im) in enumerate(exact_snr()):
        lines.append(f"{n} {re} {im}")
    Path(__file__).with_name("p7_dyadic.txt").write_text("\n".join(lines) + "\n")
