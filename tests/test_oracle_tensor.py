"""Pins of the tensor-mode oracle (reading R27: flat-space tensor line-of-sight kernels of Zaldarriaga &
Seljak 1997 Eq. 30, the forms the paper refers to at PAPER.md:54 and PAPER.md:331 without printing them)
and of the source interpolation in k (reading R26, PAPER.md:131 `InterpolateSources`).  None of these
re-types the oracle's own formulas:

  T1  j_l' and j_l'' against 40-digit mpmath derivatives of sqrt(pi/2x) J_{l+1/2}(x);
  T2  sum rules  sum_l (2l+1) j_l'(x)^2 = 1/3  and  sum_l (2l+1) j_l(x) j_l'(x) = 0  (derivatives of the
      addition theorem sum (2l+1) j_l^2 = 1): a wrong sign or index in the derivative formula breaks them;
  T3  single-tau sources: Delta^X_l(k) is the radial kernel itself, compared with the kernels written out
      from mpmath's j_l, j_l', j_l'' (pins 1/x^2, the prefactor, the signs and weights of the E and B kernels);
  T4  tensor TT plateau: a single-tau unit source and P_t = 1 give C_l^TT / 4 pi -> (4/15)/((l+3)(l-2))
      (Weber-Schafheitlin, the integral behind pin P5);
  T5  the B kernel vanishes identically for no l, but E and B are orthogonal in the sense that swapping the
      sources changes the output: linearity and source separation;
  T6  C_l of Delta = 1 is 4 pi ln(k_max/k_min) in all four spectra, order TT, EE, BB, TE.
  S1  interp_sources: linear-in-k sources exactly; knots reproduced; scipy natural CubicSpline; columns
      (tau) independent.
"""
import mpmath as mp
import numpy as np
import pytest
from scipy.interpolate import CubicSpline

import oracle

REALS = ["f64", "f80"]
mp.mp.dps = 40


def jl_mp(l, x):
    x = mp.mpf(x)
    return mp.sqrt(mp.pi / (2 * x)) * mp.besselj(l + mp.mpf(1) / 2, x)


def kernels_mp(l, x):
    """(T, E, B) radial kernels from mpmath's j_l and its numerical derivatives."""
    j = jl_mp(l, x)
    d1 = mp.diff(lambda t: jl_mp(l, t), x)
    d2 = mp.diff(lambda t: jl_mp(l, t), x, 2)
    x = mp.mpf(x)
    pref = mp.sqrt(mp.mpf((l + 2) * (l + 1) * l * (l - 1)))
    return (pref * j / x ** 2, -j + d2 + 2 * j / x ** 2 + 4 * d1 / x, 2 * d1 + 4 * j / x)


@pytest.mark.parametrize("real", REALS)
def test_t1_derivatives_against_mpmath(real):
    for x in (0.3, 2.0, 7.3, 41.7, 150.2):
        lmax = 40
        d = oracle.sph_bessel_derivs(x, lmax, real=real)
        for l in (1, 2, 3, 7, 20, 40):
            ref = [jl_mp(l, x), mp.diff(lambda t: jl_mp(l, t), x), mp.diff(lambda t: jl_mp(l, t), x, 2)]
            env = max(abs(float(r)) for r in ref)
            for q in range(3):
                assert abs(d[q, l] - float(ref[q])) <= 5e-13 * max(env, 1e-300) * max(1.0, x), (x, l, q)


@pytest.mark.parametrize("real", REALS)
@pytest.mark.parametrize("x", [0.5, 3.0, 25.0, 400.0, 3000.0])
def test_t2_sum_rules_of_the_derivative(real, x):
    lmax = oracle.lcut(x) + 10
    d = oracle.sph_bessel_derivs(x, lmax, real=real)
    l = np.arange(lmax + 1)
    # l = 0 row carries j_0' = -j_1
    assert abs(np.sum((2 * l + 1) * d[1] ** 2) - 1.0 / 3.0) <= 2e-13 * max(1.0, x)
    assert abs(np.sum((2 * l + 1) * d[0] * d[1])) <= 2e-13 * max(1.0, x)
    # the defining equation, with the second derivative taken from the sum rule's other derivative:
    # sum (2l+1) (j_l'^2 + j_l j_l'') = 0
    assert abs(np.sum((2 * l + 1) * (d[1] ** 2 + d[0] * d[2]))) <= 4e-13 * max(1.0, x)


@pytest.mark.parametrize("real", REALS)
def test_t3_single_tau_sources_give_the_radial_kernels(real):
    tau0 = 14000.0
    tau = np.array([100.0, 280.0, 5000.0, 9000.0, 13990.0])
    i_star = 2
    chi = tau0 - tau[i_star]
    k = np.array([2.0e-4, 1.3e-3, 4.1e-3, 9.7e-3, 1.6e-2])
    w = oracle.trapz_weights(tau, real=real)
    S = np.zeros((k.size, tau.size))
    S[:, i_star] = 1.0 / w[i_star]
    Z = np.zeros_like(S)
    l_list = np.array([2, 3, 5, 17, 60, 120], dtype=np.int32)
    D_T = oracle.transfer_tensor(l_list, k, tau, tau0, S, Z, Z, real=real)
    D_E = oracle.transfer_tensor(l_list, k, tau, tau0, Z, S, Z, real=real)
    D_B = oracle.transfer_tensor(l_list, k, tau, tau0, Z, Z, S, real=real)
    # source separation: a source feeds its own transfer function only
    assert np.all(D_T[1:] == 0) and np.all(D_E[[0, 2]] == 0) and np.all(D_B[:2] == 0)
    for a, l in enumerate(l_list):
        for j, kk in enumerate(k):
            x = kk * chi
            ref = [float(v) for v in kernels_mp(int(l), x)]
            got = (D_T[0, a, j], D_E[1, a, j], D_B[2, a, j])
            for q in range(3):
                scale = max(abs(ref[q]), 1e-30)
                if abs(ref[q]) < 1e-28:        # below the R16 cut the oracle returns exact zeros
                    assert abs(got[q]) < 1e-27
                else:
                    assert abs(got[q] - ref[q]) <= 2e-11 * scale, (l, x, q, got[q], ref[q])


@pytest.mark.parametrize("real", REALS)
def test_t4_tensor_tt_plateau(real):
    """TT tensor kernel = the scalar E kernel: int (l+2)!/(l-2)! j_l^2 / x^4 dln x = (4/15)/((l+3)(l-2))."""
    tau0, chi = 14000.0, 13720.0
    tau = np.array([tau0 - chi - 50.0, tau0 - chi, tau0 - chi + 50.0])
    w = oracle.trapz_weights(tau, real=real)
    for l in (3, 5, 10, 30):
        x = np.geomspace(1e-3, 100.0 * l, 20000)
        k = x / chi
        S = np.zeros((k.size, 3))
        S[:, 1] = 1.0 / w[1]
        Z = np.zeros_like(S)
        D = oracle.transfer_tensor(np.array([l], dtype=np.int32), k, tau, tau0, S, Z, Z, real=real)
        C = oracle.cls_tensor(k, D, np.ones_like(k), real=real)
        assert abs(C[0, 0] / (4 * np.pi) / ((4.0 / 15.0) / ((l + 3) * (l - 2))) - 1.0) < 1e-4
        assert np.all(C[1:, 0] == 0)


@pytest.mark.parametrize("real", REALS)
def test_t5_linearity_and_l_subset(real):
    rng = np.random.default_rng(3)
    tau0 = 14000.0
    tau = np.sort(rng.uniform(100.0, 13900.0, 25))
    k = np.geomspace(1e-4, 2e-2, 9)
    S = [rng.standard_normal((k.size, tau.size)) for _ in range(6)]
    l_list = np.arange(2, 90, dtype=np.int32)
    D1 = oracle.transfer_tensor(l_list, k, tau, tau0, S[0], S[1], S[2], real=real)
    D2 = oracle.transfer_tensor(l_list, k, tau, tau0, S[3], S[4], S[5], real=real)
    D12 = oracle.transfer_tensor(l_list, k, tau, tau0, S[0] + 2 * S[3], S[1] + 2 * S[4], S[2] + 2 * S[5], real=real)
    assert np.max(np.abs(D12 - (D1 + 2 * D2))) <= 1e-12 * np.max(np.abs(D12))
    sub = l_list[::7]
    Ds = oracle.transfer_tensor(sub, k, tau, tau0, S[0], S[1], S[2], real=real)
    assert np.array_equal(Ds, D1[:, ::7, :])


@pytest.mark.parametrize("real", REALS)
def test_t6_cls_tensor_of_unit_transfer_functions(real):
    k = np.geomspace(1e-5, 0.3, 777)
    D = np.ones((3, 4, k.size))
    D[1] *= 2.0
    D[2] *= -3.0
    C = oracle.cls_tensor(k, D, np.ones_like(k), real=real)
    base = 4 * np.pi * np.log(k[-1] / k[0])
    for q, f in enumerate((1.0, 4.0, 9.0, 2.0)):      # TT, EE, BB, TE
        assert np.max(np.abs(C[q] / (f * base) - 1.0)) < 1e-13


# --------------------------------------------------------------------------- interpolation of the sources in k
@pytest.mark.parametrize("real", REALS)
def test_s1_interp_sources(real):
    rng = np.random.default_rng(11)
    kc = np.sort(np.concatenate([[1e-4, 0.3], rng.uniform(1e-4, 0.3, 38)]))
    k = np.sort(np.concatenate([kc[[0, 5, -1]], rng.uniform(kc[0], kc[-1], 200)]))
    n_tau = 7
    # linear in k: reproduced exactly (natural end conditions)
    a, b = rng.standard_normal(n_tau), rng.standard_normal(n_tau)
    lin = a[None, :] + b[None, :] * kc[:, None]
    out = oracle.interp_sources(kc, k, lin, real=real)
    assert np.max(np.abs(out - (a[None, :] + b[None, :] * k[:, None]))) <= 2e-15 * np.max(np.abs(lin))
    # smooth oscillating sources: scipy's natural spline (an independent library routine), knots reproduced
    S = np.cos(40.0 * kc[:, None] * (1.0 + np.arange(n_tau)[None, :])) * np.exp(-(kc[:, None] / 0.2) ** 2)
    out = oracle.interp_sources(kc, k, S, real=real)
    ref = CubicSpline(kc, S, axis=0, bc_type="natural")(k)
    assert np.max(np.abs(out - ref)) <= 1e-12
    knots = oracle.interp_sources(kc, kc, S, real=real)
    assert np.max(np.abs(knots - S)) <= 1e-15
    # the tau columns are independent
    one = oracle.interp_sources(kc, k, np.ascontiguousarray(S[:, 3:4]), real=real)
    assert np.array_equal(one[:, 0], out[:, 3])


def test_tensor_and_interp_bad_arguments():
    k = np.array([1e-3, 2e-3]); tau = np.array([1.0, 2.0]); S = np.zeros((2, 2))
    with pytest.raises(ValueError):
        oracle.transfer_tensor(np.array([2], dtype=np.int32), k, np.array([1.0, 15000.0]), 14000.0, S, S, S)
    with pytest.raises(ValueError):
        oracle.interp_sources(np.array([1.0, 2.0]), np.array([0.5]), np.zeros((2, 1)))
    with pytest.raises(ValueError):
        oracle.interp_sources(np.array([2.0, 1.0]), np.array([1.5]), np.zeros((2, 1)))
