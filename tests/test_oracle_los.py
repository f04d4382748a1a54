"""Pins P2-P9 for the oracle's transfer functions and C_l (oracle/los_oracle.c).

External truths: exact integrals of linear functions (trapezoid rule); a single-tau source
collapses Eq. 2-3 to one kernel value, checked against 50-digit mpmath (this also pins the
index order of S and Delta, the 1/x^2 and the sqrt((l+2)!/(l-2)!) of Delta^E); the
Weber-Schafheitlin integral  int_0^inf J_nu(t)^2 t^-lam dt  (A&S 11.4.33 / Watson 13.41) gives
closed forms for int j_l^2 x^-p dln x: 1/(2l(l+1)) (p=0, the Sachs-Wolfe plateau BJ names),
(4/15)/((l+3)(l-2)) (EE) and (1/3)/sqrt((l+2)(l+1)l(l-1)) (TE); C_l of Delta = 1 is
4 pi ln(k_max/k_min); Cauchy-Schwarz.
"""
import math
import os

import mpmath as mp
import numpy as np
import pytest

import oracle
from paper_2509_25110_b200 import synth

mp.mp.dps = 50
REALS = ("f64", "f80")


def _jl(l, x):
    x = mp.mpf(x)
    return mp.besselj(l + mp.mpf(1) / 2, x) * mp.sqrt(mp.pi / (2 * x))


def weber_schafheitlin(l, p):
    """int_0^inf j_l(x)^2 x^-p dx/x = (pi/2) int J_{l+1/2}(t)^2 t^-(p+2) dt, closed form."""
    lam, nu = p + 2.0, l + 0.5
    lg = math.lgamma
    val = lg(lam) + lg(nu + (1 - lam) / 2) - lam * math.log(2) - 2 * lg((1 + lam) / 2) - lg(nu + (1 + lam) / 2)
    return 0.5 * math.pi * math.exp(val)


def test_weber_schafheitlin_reduces_to_the_quoted_closed_forms():
    for l in (3, 7, 40):
        assert weber_schafheitlin(l, 0) == pytest.approx(1 / (2 * l * (l + 1)), rel=1e-12)
        pref2 = (l + 2) * (l + 1) * l * (l - 1)
        assert pref2 * weber_schafheitlin(l, 4) == pytest.approx((4 / 15) / ((l + 3) * (l - 2)), rel=1e-12)
        assert math.sqrt(pref2) * weber_schafheitlin(l, 2) == pytest.approx(1 / (3 * math.sqrt(pref2)), rel=1e-12)


# ----------------------------------------------------------------------------- P2
@pytest.mark.parametrize("real", REALS)
def test_p2_trapezoid_weights_integrate_linear_functions_exactly(real):
    t = synth.tau_grid(200, 100)
    w = oracle.trapz_weights(t, real=real)
    assert np.all(w > 0)
    assert math.fsum(w) == pytest.approx(t[-1] - t[0], rel=2e-16)
    a, b = 0.3, -2.5e-4
    exact = a * (t[-1] - t[0]) + 0.5 * b * (t[-1] ** 2 - t[0] ** 2)
    assert math.fsum(w * (a + b * t)) == pytest.approx(exact, rel=1e-14)
    # a piecewise-linear "hat" with its kink on a node is integrated exactly as well
    hat = np.maximum(0.0, 1.0 - np.abs(t - t[150]) / (t[170] - t[150]))
    hat[:150] = np.maximum(0.0, 1.0 - (t[150] - t[:150]) / (t[150] - t[120]))
    assert math.fsum(w * hat) == pytest.approx(0.5 * (t[170] - t[120]), rel=1e-14)
    w3 = oracle.trapz_weights([1.0, 2.0, 7.0], real=real)
    assert list(w3) == [0.5, 3.0, 2.5]


# ----------------------------------------------------------------------------- P3 / P6
def _single_tau_problem(n_k=7, with_phi=True):
    tau = np.array([100.0, 280.0, 700.0, 13000.0])   # w_1 = (700 - 100)/2 = 300
    tau0, istar, wstar = 14000.0, 1, 300.0
    k = np.geomspace(2e-4, 0.05, n_k)
    amp_T = 1.0 + np.arange(n_k)                      # k-dependent amplitudes pin the index order
    amp_E = 0.5 - 0.1 * np.arange(n_k)
    amp_P = 3.0 + 0.25 * np.arange(n_k) ** 2
    S_T = np.zeros((n_k, tau.size)); S_E = np.zeros_like(S_T); S_P = np.zeros_like(S_T)
    S_T[:, istar] = amp_T / wstar
    S_E[:, istar] = amp_E / wstar
    S_P[:, istar] = amp_P / wstar
    return tau, tau0, istar, k, (amp_T, amp_E, amp_P), (S_T, S_E, S_P if with_phi else None)


@pytest.mark.parametrize("real", REALS)
def test_p3_single_tau_source_gives_the_kernel_itself(real):
    tau, tau0, istar, k, amps, (S_T, S_E, S_P) = _single_tau_problem()
    l_list = np.array([2, 3, 4, 5, 9, 17, 40, 120, 300, 699], dtype=np.int32)
    D = oracle.transfer(l_list, k, tau, tau0, S_T, S_E, S_P, real=real)
    assert D.shape == (3, l_list.size, k.size)
    chi = tau0 - tau[istar]
    for a, l in enumerate(l_list):
        for j in range(k.size):
            x = float(k[j] * chi)
            jl = _jl(int(l), x)
            pref = mp.sqrt(mp.mpf(int(l) + 2) * (int(l) + 1) * int(l) * (int(l) - 1))
            want = [amps[0][j] * jl, amps[1][j] * pref * jl / mp.mpf(x) ** 2, amps[2][j] * jl]
            for s in range(3):
                scale = max(abs(float(want[s])), abs(float(want[s] / jl)) * 1e-3 / max(x, 1.0))
                assert abs(float(mp.mpf(float(D[s, a, j])) - want[s])) <= 2e-13 * scale, (s, l, j)


@pytest.mark.parametrize("real", REALS)
def test_p3_linearity_and_subset_consistency(real):
    cfg = synth.CONFIGS[0]
    ks = slice(180, 260, 9)
    S_T, S_E, _ = synth.sources(cfg, k_slice=ks)
    k, tau = cfg.k()[ks], cfg.tau()
    l_all = np.arange(2, 81, dtype=np.int32)
    D = oracle.transfer(l_all, k, tau, cfg.tau0, S_T, S_E, real=real)
    # l subset: same numbers
    sub = np.array([2, 10, 11, 57, 80], dtype=np.int32)
    Ds = oracle.transfer(sub, k, tau, cfg.tau0, S_T, S_E, real=real)
    assert np.array_equal(Ds, D[:, sub - 2, :])
    # k subset: same numbers
    Dk = oracle.transfer(l_all, k[2:5], tau, cfg.tau0, S_T[2:5], S_E[2:5], real=real)
    assert np.array_equal(Dk, D[:, :, 2:5])
    # linearity in S, sources independent of each other
    rng = np.random.default_rng(3)
    A, B = rng.standard_normal(S_T.shape), rng.standard_normal(S_T.shape)
    DA = oracle.transfer(l_all, k, tau, cfg.tau0, A, B, real=real)
    DB = oracle.transfer(l_all, k, tau, cfg.tau0, B, A, real=real)
    DAB = oracle.transfer(l_all, k, tau, cfg.tau0, 2.0 * A - 3.0 * B, 2.0 * B - 3.0 * A, real=real)
    ref = np.max(np.abs(DA), axis=2, keepdims=True) + np.max(np.abs(DB), axis=2, keepdims=True)
    assert np.max(np.abs(DAB - (2.0 * DA - 3.0 * DB)) / ref) < 1e-13
    # phi is the T code path with its own source (P6)
    DP = oracle.transfer(l_all, k, tau, cfg.tau0, A, B, S_phi=A, real=real)
    assert np.array_equal(DP[2], DP[0]) and np.array_equal(DP[:2], DA)


# ----------------------------------------------------------------------------- P4 / P5 / P6
def _plateau_cls(l_tests, x_lo, x_hi_per_l, n_k, real):
    tau = np.array([100.0, 280.0, 700.0])
    tau0, wstar = 14000.0, 300.0
    chi = tau0 - 280.0
    out = {}
    for l in l_tests:
        k = np.geomspace(x_lo, x_hi_per_l * l, n_k) / chi
        S = np.zeros((n_k, 3)); S[:, 1] = 1.0 / wstar
        D = oracle.transfer(np.array([l], dtype=np.int32), k, tau, tau0, S, S, S_phi=S, real=real)
        out[l] = oracle.cls(k, D, np.ones(n_k), real=real)[:, 0] / (4 * math.pi)
    return out


@pytest.mark.parametrize("real", REALS)
def test_p4_sachs_wolfe_plateau(real):
    """BJ: single-tau source, flat P_R => int j_l^2 dlnk = 1/(2l(l+1)) to 1e-4 on a dense k grid."""
    res = _plateau_cls((2, 5, 10, 30, 50, 100), 1e-3, 100.0, 20000, real)
    for l, c in res.items():
        want = 1.0 / (2 * l * (l + 1))
        assert c[0] == pytest.approx(want, rel=1e-4), l       # TT
        assert c[3] == pytest.approx(want, rel=1e-4), l       # phiphi: same path (P6)
        # adding the analytic tail  int_{x_hi}^inf j_l^2 dlnx ~ 1/(4 x_hi^2)  closes the gap
        assert c[0] + 1.0 / (4 * (100.0 * l) ** 2) == pytest.approx(want, rel=1e-5), l


@pytest.mark.parametrize("real", REALS)
def test_p5_ee_te_weber_schafheitlin(real):
    res = _plateau_cls((3, 5, 10, 30), 1e-4, 50.0, 40000, real)
    for l, c in res.items():
        assert c[1] == pytest.approx((4 / 15) / ((l + 3) * (l - 2)), rel=2e-6), l
        assert c[2] == pytest.approx((1 / 3) / math.sqrt((l + 2) * (l + 1) * l * (l - 1)), rel=2e-6), l


# ----------------------------------------------------------------------------- P7
@pytest.mark.parametrize("real", REALS)
def test_p7_cls_reduction(real):
    cfg = synth.CONFIGS[0]
    k = cfg.k()
    n_l = 5
    C = oracle.cls(k, np.ones((3, n_l, k.size)), np.ones(k.size), real=real)
    assert C.shape == (4, n_l)
    assert np.allclose(C, 4 * math.pi * math.log(k[-1] / k[0]), rtol=1e-14, atol=0)
    # P_R and the TE cross term: Delta^T = a, Delta^E = b constant in k, P_R = k^2 -> exact trapezoid in ln k
    rng = np.random.default_rng(11)
    D = rng.standard_normal((2, n_l, k.size))
    P = synth.primordial_power(cfg)
    C = oracle.cls(k, D, P, real=real)
    assert C.shape == (3, n_l)
    lk = np.log(k)
    w = np.empty_like(k); w[0] = (lk[1] - lk[0]) / 2; w[-1] = (lk[-1] - lk[-2]) / 2; w[1:-1] = (lk[2:] - lk[:-2]) / 2
    for a in range(n_l):
        tt = 4 * math.pi * math.fsum(w * P * D[0, a] ** 2)
        ee = 4 * math.pi * math.fsum(w * P * D[1, a] ** 2)
        te = 4 * math.pi * math.fsum(w * P * D[0, a] * D[1, a])
        assert C[0, a] == pytest.approx(tt, rel=1e-13) and C[1, a] == pytest.approx(ee, rel=1e-13)
        assert abs(C[2, a] - te) <= 1e-13 * math.sqrt(tt * ee)
    assert np.all(C[0] >= 0) and np.all(C[1] >= 0)
    assert np.all(np.abs(C[2]) <= np.sqrt(C[0] * C[1]) * (1 + 1e-14))
    # scaling: C ~ A_s, and TE flips sign with Delta^E
    D2 = D.copy(); D2[1] *= -1
    C2 = oracle.cls(k, D2, 3.0 * P, real=real)
    assert np.allclose(C2[0], 3 * C[0], rtol=1e-14) and np.allclose(C2[2], -3 * C[2], rtol=1e-14)


# ----------------------------------------------------------------------------- P8 / P9
def test_p8_skip_rule_margin_and_p9_f64_vs_f80_on_config0():
    cfg = synth.CONFIGS[0]
    S_T, S_E, _ = synth.sources(cfg)
    args = (cfg.l_list(), cfg.k(), cfg.tau(), cfg.tau0, S_T, S_E)
    D0 = oracle.transfer(*args, margin=0)
    D60 = oracle.transfer(*args, margin=60)
    D80 = oracle.transfer(*args, real="f80")
    ref = np.max(np.abs(D80), axis=2, keepdims=True)
    assert np.max(np.abs(D0 - D60) / ref) < 2e-14
    assert np.max(np.abs(D60 - D80) / ref) < 5e-14
    P = synth.primordial_power(cfg)
    C64, C80 = oracle.cls(cfg.k(), D60, P), oracle.cls(cfg.k(), D80, P, real="f80")
    assert np.max(np.abs(C64[:2] / C80[:2] - 1)) < 1e-12
    assert np.max(np.abs(C64[2] - C80[2]) / np.sqrt(C80[2] ** 2 + C80[0] * C80[1])) < 1e-12   # R13
    assert np.all(np.abs(C80[2]) <= np.sqrt(C80[0] * C80[1]))


def test_bad_arguments():
    cfg = synth.CONFIGS[0]
    S = np.zeros((2, cfg.n_tau))
    with pytest.raises(ValueError):
        oracle.transfer(cfg.l_list(), [-1.0, 2.0], cfg.tau(), cfg.tau0, S, S)
    with pytest.raises(ValueError):
        oracle.transfer(cfg.l_list(), [1.0, 2.0], cfg.tau(), cfg.tau()[-1], S, S)


def _survey_golden():
    rows = []
    with open(os.path.join(os.path.dirname(__file__), "golden", "config0_survey.txt")) as f:
        for line in f:
            if line.strip() and not line.startswith("#"):
                rows.append(line.split())
    return rows


def test_generator_spot_values_of_survey_a5():
    """grids and noisy sources of config 0 (libm-dependent at the ulp level: 1e-13)."""
    cfg = synth.CONFIGS[0]
    arrays = {"k": cfg.k(), "tau": cfg.tau()}
    arrays["S_T"], arrays["S_E"], _ = synth.sources(cfg)
    n = 0
    for row in _survey_golden():
        if row[0] in arrays:
            idx = tuple(int(v) for v in row[1:-1])
            assert arrays[row[0]][idx] == pytest.approx(float(row[-1]), rel=1e-13)
            n += 1
    assert n == 7


@pytest.mark.parametrize("real", REALS)
def test_p9_config0_spectra_against_the_surveys_independent_prototype(real):
    """C_l of config 0 from an implementation written before and without this
    oracle (numpy long double, all-downward recurrence).  Pins the whole pipeline -- grids, weights,
    Bessel columns, Delta^E prefactor and 1/x^2, ln k weights, 4 pi -- at config 0 to the 12 printed
    digits (TE relative to sqrt(TE^2 + TT EE), reading R13: it crosses zero between l = 100 and 150)."""
    cfg = synth.CONFIGS[0]
    S_T, S_E, _ = synth.sources(cfg)
    D = oracle.transfer(cfg.l_list(), cfg.k(), cfg.tau(), cfg.tau0, S_T, S_E, real=real)
    C = oracle.cls(cfg.k(), D, synth.primordial_power(cfg), real=real)
    n = 0
    for row in _survey_golden():
        if row[0] == "cl":
            a = int(row[1]) - cfg.l_min
            tt, ee, te = (float(v) for v in row[2:])
            assert C[0, a] == pytest.approx(tt, rel=2e-12)
            assert C[1, a] == pytest.approx(ee, rel=2e-12)
            assert abs(C[2, a] - te) <= 2e-12 * np.sqrt(te * te + tt * ee)
            n += 1
    assert n == 7
