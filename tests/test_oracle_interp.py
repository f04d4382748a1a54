"""Pins of oracle.cl_interp (reading R25: natural cubic spline of l(l+1) C_l in l; the paper names
"spline interpolation" between the "explicitly computed multipoles", without
defining it).  None of these re-types the oracle's formulas:
  P10a  data on a straight line in y = l(l+1) C_l are reproduced exactly (a natural spline reproduces
        linear functions and nothing of higher degree: its end conditions force s'' = 0);
  P10b  the sampled multipoles are returned unchanged;
  P10c  agreement with scipy.interpolate.CubicSpline(bc_type="natural"), an independent library routine;
  P10d  C^2: the second differences of y on the integer grid have no jump at the knots beyond the
        cubic's own third-derivative step;
  P10e  a smooth spectrum sampled like CAMB's default (every l at low l, every 50th above) is recovered
        to the known O(h^4) accuracy: 16x smaller error when the spacing halves;
  P10f  config 0: the all-l oracle spectra from a 29-point l list, to a stated accuracy.
"""
import numpy as np
import pytest
from scipy.interpolate import CubicSpline

import oracle
from paper_2509_25110_b200 import synth


def camb_like_list(l_min, l_max, dense_to=40, step_mid=10, mid_to=200, step_hi=50):
    l = np.concatenate([np.arange(l_min, dense_to), np.arange(dense_to, mid_to, step_mid),
                        np.arange(mid_to, l_max + 1, step_hi), [l_max]])
    return np.unique(l[(l >= l_min) & (l <= l_max)]).astype(np.int32)


@pytest.mark.parametrize("real", ["f64", "f80"])
def test_linear_data_are_reproduced_exactly(real):
    l_list = np.array([2, 3, 5, 9, 20, 50, 51, 120, 400], dtype=np.int32)
    l_all = np.arange(2, 401)
    a, b = 3.5e-10, 2.25e-12
    y = a + b * l_list                                   # y = l(l+1) C_l on a straight line
    C = oracle.cl_interp(l_list, (y / (l_list * (l_list + 1.0)))[None, :], real=real)[0]
    want = (a + b * l_all) / (l_all * (l_all + 1.0))
    assert np.max(np.abs(C / want - 1.0)) < 5e-15


def test_knots_are_returned_unchanged_and_rows_are_independent():
    rng = np.random.default_rng(3)
    l_list = camb_like_list(2, 900)
    Cs = rng.uniform(0.5, 2.0, (4, l_list.size)) * 1e-10 / (l_list * (l_list + 1.0))
    C = oracle.cl_interp(l_list, Cs)
    assert C.shape == (4, 899)
    assert np.max(np.abs(C[:, l_list - 2] / Cs - 1.0)) < 4e-16
    C1 = oracle.cl_interp(l_list, Cs[2:3])
    assert np.array_equal(C1[0], C[2])


@pytest.mark.parametrize("real", ["f64", "f80"])
def test_against_scipy_natural_cubic_spline(real):
    rng = np.random.default_rng(11)
    for l_list in (camb_like_list(2, 2500), np.array([2, 7], dtype=np.int32), np.array([30, 31, 64], dtype=np.int32),
                   np.sort(rng.choice(np.arange(2, 3000), 80, replace=False)).astype(np.int32)):
        y = np.cos(l_list / 70.0) * np.exp(-l_list / 900.0) + 0.3 * rng.standard_normal(l_list.size)
        l_all = np.arange(l_list[0], l_list[-1] + 1)
        want = CubicSpline(l_list.astype(float), y, bc_type="natural")(l_all.astype(float))
        C = oracle.cl_interp(l_list, (y / (l_list * (l_list + 1.0)))[None, :], real=real)[0]
        got = C * (l_all * (l_all + 1.0))
        assert np.max(np.abs(got - want)) < 2e-12 * np.max(np.abs(y))


def test_second_derivative_is_continuous_at_the_knots():
    l_list = np.array([2, 12, 40, 90, 200, 420], dtype=np.int32)
    y = np.array([1.0, -2.0, 0.5, 3.0, -1.0, 2.0])
    l_all = np.arange(2, 421)
    s = oracle.cl_interp(l_list, (y / (l_list * (l_list + 1.0)))[None, :], real="f80")[0] * (l_all * (l_all + 1.0))
    d2 = s[2:] - 2 * s[1:-1] + s[:-2]                    # exact s'' at the centre point for a cubic
    d3 = np.diff(d2)                                     # piecewise constant: s''' per segment
    for kn in l_list[1:-1]:
        i = kn - 2                                        # index of the knot in l_all; d2[i-1] is centred on it
        # across a knot the second difference changes by at most one third-derivative step of either side
        assert abs(d2[i] - d2[i - 2]) <= 2.0 * max(abs(d3[i - 3]), abs(d3[i + 1])) * 1.0000001 + 1e-13
    assert abs(d2[0]) < 0.2 * np.max(np.abs(d2)) and abs(d2[-1]) < 0.2 * np.max(np.abs(d2))   # natural ends


def test_fourth_order_convergence_on_a_smooth_spectrum():
    f = lambda l: 1e-9 * (1.0 + 0.6 * np.cos(l / 95.0)) * np.exp(-(l / 1400.0) ** 2)      # y = l(l+1) C_l
    l_all = np.arange(200, 2201)
    errs = []
    for step in (80, 40, 20):
        l_list = np.arange(200, 2201, step).astype(np.int32)
        C = oracle.cl_interp(l_list, (f(l_list) / (l_list * (l_list + 1.0)))[None, :])[0]
        inner = (l_all > 600) & (l_all < 1800)            # away from the natural ends (their error is O(h^2))
        errs.append(np.max(np.abs(C * l_all * (l_all + 1.0) - f(l_all))[inner]))
    assert 11.0 < errs[0] / errs[1] < 21.0 and 11.0 < errs[1] / errs[2] < 21.0
    # the classical bound |f - s| <= 5/384 h^4 max|f| (Hall & Meyer 1976), f by central differences
    x = np.arange(200.0, 2200.5, 0.5)
    f4 = (f(x[4:]) - 4 * f(x[3:-1]) + 6 * f(x[2:-2]) - 4 * f(x[1:-3]) + f(x[:-4])) / 0.5 ** 4
    assert errs[2] <= 5.0 / 384.0 * 20.0 ** 4 * np.max(np.abs(f4))
    assert errs[2] >= 1e-3 * 5.0 / 384.0 * 20.0 ** 4 * np.max(np.abs(f4))      # and it is not trivially zero


def test_config0_spectra_from_a_sparse_l_list():
    """BASELINE.json config 0 (l = 2..200) end to end on the oracle side: transfer functions on 55 of the
    199 multipoles only (every l below 20, every 5th above), their spectra, then the spline, against the
    all-l oracle spectra.  The knots come back exactly; in between the synthetic spectrum limits the
    accuracy, not the spline: config 0's 400-point k grid undersamples Delta_l(k) above k ~ 0.01, which
    leaves an l-to-l jitter of a few per cent in C_l at l > 100 that no interpolation can follow
    (halving the spacing does not reduce the error there).  Stated accuracy of reading R25 on this
    input: TT within 1 % up to l = 130, every spectrum within 6 % of its local level everywhere."""
    cfg = synth.CONFIGS[0]
    S_T, S_E, _ = synth.sources(cfg)
    P = synth.primordial_power(cfg)
    l_sparse = camb_like_list(2, 200, dense_to=20, step_mid=5, mid_to=200, step_hi=50)
    assert l_sparse.size == 55
    l_all = cfg.l_list()
    D_all = oracle.transfer(l_all, cfg.k(), cfg.tau(), cfg.tau0, S_T, S_E)
    C_all = oracle.cls(cfg.k(), D_all, P)
    D_sp = oracle.transfer(l_sparse, cfg.k(), cfg.tau(), cfg.tau0, S_T, S_E)
    assert np.array_equal(D_sp, D_all[:, l_sparse - 2, :])        # l-subset consistency (P3)
    C_sp = oracle.cls(cfg.k(), D_sp, P)
    C_int = oracle.cl_interp(l_sparse, C_sp)
    assert C_int.shape == C_all.shape
    assert np.max(np.abs(C_int[:, l_sparse - 2] / C_sp - 1.0)) < 4e-16
    assert np.max(np.abs(C_int[0] / C_all[0] - 1.0)[l_all <= 130]) < 1e-2
    for q in (0, 1):
        assert np.max(np.abs(C_int[q] / C_all[q] - 1.0)) < 6e-2
    norm = np.sqrt(C_all[2] ** 2 + C_all[0] * C_all[1])
    assert np.max(np.abs(C_int[2] - C_all[2]) / norm) < 6e-2
