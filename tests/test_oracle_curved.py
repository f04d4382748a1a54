"""Pins of the open-universe oracle (reading R28: hyperspherical Bessel functions,
PAPER.md:60, 250, 258).  The paper prints no formula, so the first pin goes back to first principles:

  H0  the 60-digit mpmath FORWARD recurrence used as reference below satisfies the radial Helmholtz
      equation of hyperbolic space  Phi'' + 2 coth(chi) Phi' + [beta^2 + 1 - l(l+1)/sinh^2(chi)] Phi = 0
      and starts from Phi_0 = sin(beta chi)/(beta sinh chi): it IS the function R28 names;
  H1  the oracle (Miller's DOWNWARD recurrence in fp64 / x87) against that reference, below and above the
      turning point (150 digits keep the forward direction accurate there);
  H2  flat limit: Phi_l^beta(x/beta) -> j_l(x) as beta -> infinity, with an error that falls like 1/beta^2;
  H3  skip rule: |Phi_l| < 1e-30 at the oracle's curved-space cut, where the flat formula L_cut(beta sinh chi)
      would still be at 1e-19 ... 1e-6;
  H4  transfer functions: single-tau sources give Phi_l(chi*) and, for E, sqrt((l+2)!/(l-2)!) Phi_l/(beta
      sinh chi*)^2; K -> 0 reproduces the flat oracle; linearity.
"""
import mpmath as mp
import numpy as np
import pytest

import oracle

REALS = ["f64", "f80"]


def phi_forward(lmax, beta, chi):
    beta, chi = mp.mpf(beta), mp.mpf(chi)
    b = lambda l: mp.sqrt(beta ** 2 + l ** 2)
    out = [mp.sin(beta * chi) / (beta * mp.sinh(chi))]
    out.append((mp.coth(chi) * mp.sin(beta * chi) - beta * mp.cos(beta * chi)) / (beta * mp.sinh(chi) * b(1)))
    for l in range(2, lmax + 1):
        out.append(((2 * l - 1) * mp.coth(chi) * out[l - 1] - b(l - 1) * out[l - 2]) / b(l))
    return out


def test_h0_the_reference_satisfies_the_radial_equation():
    mp.mp.dps = 60
    for beta, chi in ((37.3, 0.41), (3.0, 1.7), (0.5, 0.9)):
        beta, chi = mp.mpf(beta), mp.mpf(chi)
        for l in (0, 1, 2, 5, 11):
            f = lambda c: phi_forward(l, beta, c)[l]
            res = mp.diff(f, chi, 2) + 2 * mp.coth(chi) * mp.diff(f, chi) + \
                (beta ** 2 + 1 - l * (l + 1) / mp.sinh(chi) ** 2) * f(chi)
            assert abs(res) < mp.mpf(10) ** -40 * (1 + beta ** 2)
    # regular at the origin: Phi_l -> prod_{m<=l} sqrt(beta^2+m^2)/beta^l (beta chi)^l / (2l+1)!!
    # (the forward direction needs the digits here)
    mp.mp.dps = 150
    for l in (1, 2, 5):
        small = phi_forward(l, mp.mpf(3), mp.mpf("1e-3"))[l]
        norm = mp.fprod(mp.sqrt(9 + m * m) for m in range(1, l + 1)) / mp.mpf(3) ** l
        assert abs(small / (norm * mp.mpf("3e-3") ** l / mp.fac2(2 * l + 1)) - 1) < mp.mpf("1e-4")


@pytest.mark.parametrize("real", REALS)
def test_h1_oracle_against_the_forward_recurrence(real):
    mp.mp.dps = 150
    for beta, chi in ((37.3, 0.41), (5.0, 0.05), (200.0, 1.3), (3000.0, 0.9), (0.7, 2.0), (0.01, 0.001), (50.0, 3.0)):
        L = oracle.hyp_lcut_open(beta, chi)
        ref = phi_forward(L, beta, chi)
        got = oracle.hyp_bessel_open(beta, chi, L, real=real)
        env = max(abs(float(r)) for r in ref)
        tol = (5e-16 if real == "f64" else 2e-18) * max(1.0, beta * chi)      # neutral error growth ~ eps x
        assert max(abs(got[l] - float(ref[l])) for l in range(L + 1)) <= 200 * tol * env
        # H3: the cut lies in the negligible region (and the flat cut would not, for chi of order one)
        assert abs(ref[L]) < 1e-30
    assert abs(phi_forward(36, 0.7, 2.0)[36]) > 1e-7          # = L_cut(beta sinh chi) of the flat formula


@pytest.mark.parametrize("real", REALS)
def test_h2_flat_limit(real):
    x = 15.3
    j = oracle.sph_bessel(x, 30, real=real)
    errs = []
    for beta in (1e2, 1e3, 1e4):
        ph = oracle.hyp_bessel_open(beta, x / beta, 30, real=real)
        errs.append(np.max(np.abs(ph - j)))
    assert errs[2] < 2e-7
    assert 80 < errs[0] / errs[1] < 125 and 80 < errs[1] / errs[2] < 125      # error ~ 1/beta^2 ~ |K|


@pytest.mark.parametrize("real", REALS)
def test_h4_transfer_functions(real):
    mp.mp.dps = 150
    tau0, K = 14000.0, -(1.0 / 9000.0) ** 2
    rc = 9000.0
    tau = np.array([100.0, 280.0, 5000.0, 9000.0, 13990.0])
    i_star = 2
    k = np.array([2.0e-4, 1.3e-3, 4.1e-3, 9.7e-3])
    w = oracle.trapz_weights(tau, real=real)
    S = np.zeros((k.size, tau.size))
    S[:, i_star] = 1.0 / w[i_star]
    l_list = np.array([2, 3, 5, 17, 60, 120], dtype=np.int32)
    D = oracle.transfer_open(l_list, k, tau, tau0, K, S, S, S, real=real)
    chi = (tau0 - tau[i_star]) / rc
    for j, kk in enumerate(k):
        ref = phi_forward(int(l_list[-1]), kk * rc, chi)
        for a, l in enumerate(l_list):
            ph = float(ref[l])
            if abs(ph) < 1e-25:
                continue
            pref = np.sqrt((l + 2.0) * (l + 1.0) * l * (l - 1.0))
            bs = kk * rc * np.sinh(chi)
            assert abs(D[0, a, j] - ph) <= 1e-11 * abs(ph)
            assert abs(D[2, a, j] - ph) <= 1e-11 * abs(ph)
            assert abs(D[1, a, j] - pref * ph / bs ** 2) <= 1e-11 * abs(pref * ph / bs ** 2)
    # K -> 0: the flat oracle, with a difference that falls like |K|
    rng = np.random.default_rng(5)
    tau2 = np.sort(rng.uniform(100.0, 13900.0, 12))
    S_T, S_E = rng.standard_normal((k.size, 12)), rng.standard_normal((k.size, 12))
    l2 = np.arange(2, 60, dtype=np.int32)
    flat = oracle.transfer(l2, k, tau2, tau0, S_T, S_E, real=real)
    d = []
    for r in (1e6, 1e7):
        cur = oracle.transfer_open(l2, k, tau2, tau0, -1.0 / r ** 2, S_T, S_E, real=real)
        d.append(np.max(np.abs(cur - flat)) / np.max(np.abs(flat)))
    assert d[1] < 1e-4 and 50 < d[0] / d[1] < 200
    # linearity
    a = oracle.transfer_open(l2, k, tau2, tau0, K, S_T, S_E, real=real)
    b = oracle.transfer_open(l2, k, tau2, tau0, K, 2 * S_T, -3 * S_E, real=real)
    assert np.max(np.abs(b[0] - 2 * a[0])) <= 1e-14 * np.max(np.abs(a[0]))
    assert np.max(np.abs(b[1] + 3 * a[1])) <= 1e-14 * np.max(np.abs(a[1]))


# --------------------------------------------------------------------------- closed universes (K > 0)
def phi_forward_closed(lmax, beta, chi):
    beta, chi = mp.mpf(beta), mp.mpf(chi)
    b = lambda l: mp.sqrt(beta ** 2 - l ** 2)
    out = [mp.sin(beta * chi) / (beta * mp.sin(chi))]
    out.append((mp.cot(chi) * mp.sin(beta * chi) - beta * mp.cos(beta * chi)) / (beta * mp.sin(chi) * b(1)))
    for l in range(2, lmax + 1):
        out.append(((2 * l - 1) * mp.cot(chi) * out[l - 1] - b(l - 1) * out[l - 2]) / b(l))
    return out


def test_h0c_the_closed_reference_satisfies_the_radial_equation_of_the_three_sphere():
    """Phi'' + 2 cot(chi) Phi' + [beta^2 - 1 - l(l+1)/sin^2(chi)] Phi = 0, and the recurrence ends by itself:
    b_beta = 0, so Phi_{beta-1} is the last function (the forward recurrence gives Phi_beta = 0/0)."""
    mp.mp.dps = 60
    for beta, chi in ((40, 0.41), (7, 1.2), (12, 0.9)):
        chi = mp.mpf(chi)
        for l in (0, 1, 2, 5, 6):
            f = lambda c: phi_forward_closed(l, beta, c)[l]
            res = mp.diff(f, chi, 2) + 2 * mp.cot(chi) * mp.diff(f, chi) + \
                (mp.mpf(beta) ** 2 - 1 - l * (l + 1) / mp.sin(chi) ** 2) * f(chi)
            assert abs(res) < mp.mpf(10) ** -40 * beta ** 2
    # the numerator of the step that would give Phi_beta vanishes: (2 beta - 1) cot Phi_{beta-1} = b_{beta-1} Phi_{beta-2}
    ph = phi_forward_closed(6, 7, mp.mpf("1.2"))
    assert abs(13 * mp.cot(mp.mpf("1.2")) * ph[6] - mp.sqrt(49 - 36) * ph[5]) < mp.mpf(10) ** -50


@pytest.mark.parametrize("real", REALS)
def test_h1c_closed_oracle_against_the_forward_recurrence(real):
    mp.mp.dps = 150
    for beta, chi in ((40, 0.41), (5, 0.05), (200, 1.3), (3000, 0.9), (3, 1.5), (7, 1.2), (900, 0.002), (50, 1.5707)):
        L = oracle.hyp_lcut_closed(beta, chi)
        assert L <= beta - 1
        ref = phi_forward_closed(L, beta, chi)
        got = oracle.hyp_bessel_closed(beta, chi, beta + 3, real=real)
        env = max(abs(float(r)) for r in ref)
        tol = (5e-16 if real == "f64" else 2e-18) * max(1.0, beta * chi)
        assert max(abs(got[l] - float(ref[l])) for l in range(L + 1)) <= 200 * tol * env
        assert np.all(got[beta:] == 0.0)                       # Phi_l^beta = 0 for l >= beta
        assert L == beta - 1 or abs(ref[L]) < 1e-30            # the cut is either the end of the ladder or negligible
    # flat limit, error ~ 1/beta^2
    x = 15.3
    j = oracle.sph_bessel(x, 30, real=real)
    errs = [np.max(np.abs(oracle.hyp_bessel_closed(b, x / b, 30, real=real) - j)) for b in (100, 1000, 10000)]
    assert errs[2] < 2e-7 and 80 < errs[0] / errs[1] < 125 and 80 < errs[1] / errs[2] < 125


@pytest.mark.parametrize("real", REALS)
def test_h4c_closed_transfer_functions(real):
    mp.mp.dps = 150
    tau0, rc = 14000.0, 12000.0
    K = 1.0 / rc ** 2
    tau = np.array([100.0, 280.0, 5000.0, 9000.0, 13990.0])
    i_star = 2
    betas = np.array([3, 8, 25, 90, 200])
    k = betas / rc
    w = oracle.trapz_weights(tau, real=real)
    S = np.zeros((k.size, tau.size))
    S[:, i_star] = 1.0 / w[i_star]
    l_list = np.array([2, 3, 5, 7, 24, 25, 60, 120], dtype=np.int32)
    D = oracle.transfer_curved(l_list, k, tau, tau0, K, S, S, S, real=real)
    chi = (tau0 - tau[i_star]) / rc
    for j, beta in enumerate(betas):
        ref = phi_forward_closed(min(int(l_list[-1]), beta - 1), int(beta), chi)
        for a, l in enumerate(l_list):
            if l >= beta:
                assert D[0, a, j] == 0.0 and D[1, a, j] == 0.0 and D[2, a, j] == 0.0
                continue
            ph = float(ref[l])
            if abs(ph) < 1e-25:
                continue
            pref = np.sqrt((l + 2.0) * (l + 1.0) * l * (l - 1.0))
            bs = beta * np.sin(chi)
            assert abs(D[0, a, j] - ph) <= 1e-11 * abs(ph) and abs(D[2, a, j] - ph) <= 1e-11 * abs(ph)
            assert abs(D[1, a, j] - pref * ph / bs ** 2) <= 1e-11 * abs(pref * ph / bs ** 2)
    # non-integer beta, beta < 3 and chi > pi/2 are rejected
    for bad_k, bad_K in ((np.array([3.4, 8.0]) / rc, K), (np.array([2.0, 8.0]) / rc, K), (k, 1.0 / 5000.0 ** 2)):
        with pytest.raises(ValueError):
            oracle.transfer_curved(l_list, bad_k, tau, tau0, bad_K, S[:bad_k.size], S[:bad_k.size])


def test_curved_bad_arguments():
    k = np.array([1e-3, 2e-3]); tau = np.array([1.0, 2.0]); S = np.zeros((2, 2))
    with pytest.raises(ValueError):
        oracle.transfer_open(np.array([2], dtype=np.int32), 1.05 * k, tau, 14000.0, +1e-8, S, S)   # closed: beta = 10.5 is not an integer
    with pytest.raises(ValueError):
        oracle.hyp_bessel_open(-1.0, 0.5, 3)
