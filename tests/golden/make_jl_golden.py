"""Writes tests/golden/jl_golden.txt: spherical Bessel values j_l(x) to 25 digits.

Brute force, independent of oracle/ and of the CUDA path (mpmath only, 60 digits):
downward three-term recurrence started 200 + 5 sqrt(x) orders above max(l, x) + 20 x^(1/3),
normalised with the SUM RULE  sum_l (2l+1) j_l(x)^2 = 1  (Abramowitz & Stegun 10.1.50), i.e.
without the closed forms of j_0, j_1 that the oracle normalises with.  For x <= 50 the value is
cross-checked against mpmath's own besselj(l + 1/2, x) sqrt(pi / 2x).

The (l, x) pairs span the configs of BASELINE.json: tiny x, the turning point l ~ x, the
evanescent side x < l, the oscillatory side x > l, up to l = 10^4 and x = 16560.

Run:  python tests/golden/make_jl_golden.py
"""
import os

import mpmath as mp

mp.mp.dps = 60

PAIRS = [(0, 1.0), (1, 1.0), (2, 1.0), (10, 1.0), (5, 0.001), (3, 1e-5), (2, 3.141592653589793),
         (2, 10.0), (10, 10.0), (50, 10.0), (7, 31.4159), (100, 100.0), (200, 100.0), (90, 113.7),
         (1000, 1000.0), (1200, 1000.0), (2500, 2400.0), (2500, 2500.0), (2500, 8280.0),
         (17, 8280.0), (6000, 6000.0), (6000, 13800.0), (10000, 9990.0), (10000, 16560.0),
         (2, 16560.0)]


def column(x, lmax):
    x = mp.mpf(x)
    top = int(max(lmax, float(x)) + 20 * float(x) ** (1 / 3) + 200 + 5 * float(x) ** 0.5)
    f_hi, f = mp.mpf(0), mp.mpf(10) ** -50
    vals = {}
    norm = mp.mpf(0)
    for l in range(top, -1, -1):
        if l <= lmax:
            vals[l] = f
        norm += (2 * l + 1) * f * f
        f_hi, f = f, (2 * l + 1) / x * f - f_hi
    sign = 1 if (vals[0] > 0) == (mp.sin(x) / x > 0) else -1   # the sum rule fixes |scale| only
    sc = sign / mp.sqrt(norm)
    return {l: v * sc for l, v in vals.items()}


def main():
    lines = ["# l  x(repr of the fp64 argument)  j_l(x)   -- written by make_jl_golden.py, 60-digit mpmath"]
    for l, x in PAIRS:
        v = column(x, l)[l]
        if x <= 50:
            ref = mp.besselj(l + mp.mpf(1) / 2, mp.mpf(x)) * mp.sqrt(mp.pi / (2 * mp.mpf(x)))
            assert abs(v - ref) <= abs(ref) * mp.mpf(10) ** -40, (l, x)
        lines.append(f"{l} {x!r} {mp.nstr(v, 25)}")
    out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "jl_golden.txt")
    with open(out, "w") as fh:
        fh.write("\n".join(lines) + "\n")


if __name__ == "__main__":
    main()
