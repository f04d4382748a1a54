"""Pins P1a-P1d for the oracle's spherical-Bessel column (oracle/los_oracle.c).

Truths used (none of them is the oracle): closed forms of j_0, j_1, j_2 evaluated in 50-digit
mpmath; the sum rule sum (2l+1) j_l^2 = 1 (A&S 10.1.50); golden 60-digit values written by
tests/golden/make_jl_golden.py (sum-rule-normalised recurrence, cross-checked against
mpmath.besselj); live mpmath.besselj brute force on tiny inputs; and the cut L_cut(x) of
reading R16 checked to lie in the |j_l| < 1e-36 region.
"""
import math
import os

import mpmath as mp
import numpy as np
import pytest

import oracle

mp.mp.dps = 50
REALS = ("f64", "f80")
GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "jl_golden.txt")


def _closed(x):
    x = mp.mpf(x)
    s, c = mp.sin(x), mp.cos(x)
    return [s / x, s / x ** 2 - c / x, (3 / x ** 3 - 1 / x) * s - 3 * c / x ** 2]


def _env(x):
    """Amplitude scale of the oscillatory j_l: 1/max(x, 1)."""
    return 1.0 / max(x, 1.0)


@pytest.mark.parametrize("real", REALS)
def test_p1a_closed_forms_j0_j1_j2(real):
    rng = np.random.default_rng(7)
    xs = np.concatenate([10.0 ** rng.uniform(-5, 4.2, 300), [1e-5, 0.05, 0.999, 1.0, 1.001, math.pi,
                         2 * math.pi * (1 + 1e-13), 16560.0, 8280.0, 4116.0]])
    worst = 0.0
    for x in xs:
        got = oracle.sph_bessel(float(x), 2, real=real)
        want = _closed(float(x))
        for l in range(3):
            # neutral error growth of the recurrence: eps * x relative to the envelope 1/x
            tol = (4e-16 * max(x, 1.0) + 1e-15) * max(_env(x), abs(float(want[l])))
            err = abs(float(mp.mpf(float(got[l])) - want[l]))
            worst = max(worst, err / tol)
    assert worst < 1.0, worst


@pytest.mark.parametrize("real", REALS)
def test_p1a_relative_accuracy_small_x(real):
    # x < 1: no zeros, j_0, j_1, j_2 must be good to a few ulp RELATIVE (series branch of j_1)
    for x in (1e-5, 1e-3, 0.049, 0.051, 0.3, 0.99):
        got = oracle.sph_bessel(x, 2, real=real)
        want = _closed(x)
        for l in range(3):
            assert abs(float(mp.mpf(float(got[l])) / want[l] - 1)) < 5e-15, (x, l)


@pytest.mark.parametrize("real", REALS)
@pytest.mark.parametrize("x", [0.1, 1.0, 10.0, 100.0, 1000.0, 5000.0, 16560.0])
def test_p1b_sum_rule(real, x):
    L = oracle.lcut(x) + 30
    j = oracle.sph_bessel(x, L, real=real)
    l = np.arange(L + 1)
    assert abs(float(np.sum((2 * l + 1) * j * j)) - 1.0) < 5e-15


def _golden_rows():
    rows = []
    with open(GOLDEN) as fh:
        for line in fh:
            if line.startswith("#") or not line.strip():
                continue
            l, x, v = line.split()
            rows.append((int(l), float(x), mp.mpf(v)))
    return rows


@pytest.mark.parametrize("real", REALS)
def test_p1c_golden_values(real):
    rows = _golden_rows()
    assert len(rows) >= 20
    for l, x, want in rows:
        got = oracle.sph_bessel(x, l, real=real)[l]
        err = abs(float(mp.mpf(float(got)) - want))
        # envelope-relative 1e-12 everywhere; relative 1e-9 on the evanescent side
        assert err <= 1e-12 * max(_env(x), abs(float(want))), (l, x, got, want)
        assert err <= 1e-9 * abs(float(want)) or abs(float(want)) > 1e-6, (l, x, got, want)
        if real == "f80":
            assert err <= 2e-15 * max(_env(x), abs(float(want))), (l, x, got, want)


@pytest.mark.parametrize("real", REALS)
def test_p1d_mpmath_brute_force_tiny_inputs(real):
    worst = 0.0
    for x in (1e-5, 3e-3, 0.7, 2.5, math.pi, 9.0, 31.0, 77.7, 250.0):
        L = oracle.lcut(x)
        got = oracle.sph_bessel(x, L, real=real)
        for l in range(0, L + 1, max(1, L // 40)):
            want = mp.besselj(l + mp.mpf(1) / 2, mp.mpf(x)) * mp.sqrt(mp.pi / (2 * mp.mpf(x)))
            err = abs(float(mp.mpf(float(got[l])) - want))
            tol = 1e-13 * max(_env(x), abs(float(want))) if l <= x else 1e-12 * abs(float(want)) + 1e-300
            worst = max(worst, err / tol)
    assert worst < 1.0, worst


def test_r16_cut_is_in_the_negligible_region():
    """|j_l(x)| < 1e-36 at l = L_cut(x) (and it only decreases above): brute force in mpmath."""
    for x in (1e-5, 1e-3, 0.1, 1.0, math.pi, 10.0, 30.0, 100.0, 300.0, 1000.0):
        L = oracle.lcut(x)
        v = mp.besselj(L + mp.mpf(1) / 2, mp.mpf(x)) * mp.sqrt(mp.pi / (2 * mp.mpf(x)))
        assert abs(v) < mp.mpf(10) ** -36, (x, L, v)
        v1 = mp.besselj(L + 1 + mp.mpf(1) / 2, mp.mpf(x)) * mp.sqrt(mp.pi / (2 * mp.mpf(x)))
        assert abs(v1) < abs(v)
    # large x: brute force again (the golden script's sum-rule-normalised 60-digit recurrence)
    import importlib.util
    spec = importlib.util.spec_from_file_location(
        "make_jl_golden", os.path.join(os.path.dirname(GOLDEN), "make_jl_golden.py"))
    gold = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(gold)
    for x in (2400.0, 9990.0, 2e4):
        L = oracle.lcut(x)
        col = gold.column(x, L + 1)
        assert abs(col[L]) < mp.mpf(10) ** -36 and abs(col[L + 1]) < abs(col[L]), (x, L, col[L])


@pytest.mark.parametrize("real", REALS)
def test_zero_above_cut_and_margin_independence(real):
    x = 57.3
    L = oracle.lcut(x)
    a = oracle.sph_bessel(x, L + 80, margin=0, real=real)
    b = oracle.sph_bessel(x, L + 80, margin=60, real=real)
    assert np.all(a[L + 1:] == 0.0) and np.all(b[L + 61:] == 0.0)
    assert np.all(np.abs(b[L + 1:]) < 1e-36)
    # different start index, same function: agreement at rounding level where j_l is not negligible
    assert np.max(np.abs(a[:L + 1] - b[:L + 1])) < 5e-15 * _env(x)
    big = np.abs(b[:L + 1]) > 1e-30
    assert np.max(np.abs(a[:L + 1][big] / b[:L + 1][big] - 1)) < 1e-6


def test_f64_vs_f80_cross_check():
    for x in (0.37, 41.0, 977.0, 8280.0, 16560.0):
        L = oracle.lcut(x)
        a = oracle.sph_bessel(x, L, real="f64")
        b = oracle.sph_bessel(x, L, real="f80")
        assert np.max(np.abs(a - b)) < 2e-15 * max(x, 1.0) * _env(x) + 1e-16


def test_bad_arguments():
    with pytest.raises(ValueError):
        oracle.sph_bessel(0.0, 3)
    with pytest.raises(ValueError):
        oracle.sph_bessel(-1.0, 3)
