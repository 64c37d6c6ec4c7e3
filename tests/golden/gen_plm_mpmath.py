"""Writes tests/golden/plm_mpmath.txt: high-precision values of Pbar_lm(theta) = Y_lm(theta, 0).

Source of the values: the LIBRARY routine mpmath.spherharm (hypergeometric evaluation, 60
digits) -- not the oracle, not the CUDA path, and not a recurrence retyped here.  The
(l, m, theta) list is the one SURVEY.md 8(c) pin P5 names, plus a few near-pole and near-equator
cases.  theta is the binary64 nearest to the decimal shown, stored as a C99 hex float so the
test feeds the oracle the identical binary64.

Each line:  l  m  theta_hex  frac  exp2      with value = frac * 2**exp2, 0.5 <= |frac| < 1.

    python tests/golden/gen_plm_mpmath.py
"""
import os

import mpmath as mp

CASES = [
    (0, 0, 0.7), (1, 0, 0.7), (1, 1, 0.7), (2, 0, 2.1), (2, 1, 0.3), (2, 2, 2.9),
    (10, 3, 0.3), (33, 32, 0.05), (100, 50, 1.0), (100, 99, 3.0), (255, 0, 1e-3),
    (1000, 500, 1.0), (1000, 0, 2.0), (1000, 999, 1.5707963267948966),
    (4095, 2000, 1.0), (4095, 4095, 1.5), (4095, 4095, 0.1), (4095, 4000, 0.5),
    (4095, 1, 0.05), (4095, 0, 3.1), (4095, 300, 0.08),
    (8191, 4000, 1.0), (8191, 8191, 0.01), (8191, 8000, 1.2), (8191, 100, 0.02),
]


def main():
    mp.mp.dps = 60
    here = os.path.dirname(os.path.abspath(__file__))
    lines = ["# l m theta_hex frac exp2   (value = frac * 2**exp2; mpmath %s spherharm, 60 digits)" % mp.__version__]
    for l, m, t in CASES:
        th = mp.mpf(float(t))
        v = mp.re(mp.spherharm(l, m, th, 0, maxprec=400000, maxterms=10**6))
        frac, ex = mp.frexp(v)
        lines.append("%d %d %s %s %d" % (l, m, float(t).hex(), mp.nstr(frac, 25), ex))
    with open(os.path.join(here, "plm_mpmath.txt"), "w") as f:
        f.write("\n".join(lines) + "\n")


if __name__ == "__main__":
    main()
