"""gcamb_los_cl_interp: spectra on every multipole from spectra on a sparse l list (SURVEY 8(f)
NEXT-2; reading R25: natural cubic spline of l(l+1) C_l in l).

The CUDA kernel is compared element by element with the long-double oracle (oracle.cl_interp, pinned
in tests/test_oracle_interp.py):
  * on the oracle's own sampled spectra (isolates the spline kernel: rounding level),
  * end to end at config-1 size with a CAMB-like l list: sparse transfer -> cls -> interp on the GPU
    against the same three steps of the oracle, at the C_l bar of BASELINE.json (1e-8, reading R13),
  * batched, for ragged lists (two knots, neighbouring knots, gaps of one), and for the error paths.
"""
import numpy as np
import pytest
import torch

import oracle
from paper_2509_25110_b200 import synth

pytestmark = pytest.mark.gpu

TOL_CL = 1e-8


@pytest.fixture(scope="module")
def los():
    from paper_2509_25110_b200 import los as _los
    _los.load_library()
    assert torch.cuda.is_available()
    return _los


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def camb_like_list(l_min, l_max, dense_to=40, step_mid=10, mid_to=200, step_hi=50):
    l = np.concatenate([np.arange(l_min, dense_to), np.arange(dense_to, mid_to, step_mid),
                        np.arange(mid_to, l_max + 1, step_hi), [l_max]])
    return np.unique(l[(l >= l_min) & (l <= l_max)]).astype(np.int32)


def small_plan(los, l_list):
    k = np.geomspace(1e-4, 0.1, 8)
    tau = np.linspace(100.0, 13000.0, 40)
    return los.Plan(l_list, k, tau, 14000.0)


def interp_err(C_gpu, C_ref):
    """auto spectra relative; TE against sqrt(TE^2 + TT EE) (reading R13)"""
    e_auto = float(np.max(np.abs(C_gpu[..., :2, :] / C_ref[..., :2, :] - 1.0)))
    norm = np.sqrt(C_ref[..., 2, :] ** 2 + C_ref[..., 0, :] * C_ref[..., 1, :])
    e_te = float(np.max(np.abs(C_gpu[..., 2, :] - C_ref[..., 2, :]) / norm))
    return e_auto, e_te


@pytest.mark.parametrize("l_list", [
    [2, 9],                                        # two knots: the spline is the straight line in y
    [2, 3, 4, 5, 6],                               # every l listed: nothing to interpolate
    [5, 6, 8, 9, 40, 41, 300, 1000, 1001, 2500],   # neighbouring knots next to long gaps
    list(camb_like_list(2, 2500)),
    list(range(2, 3000, 3)),                       # 1000 knots
    list(range(2, 6500, 3)),                       # 2166 knots > 2048: the sequential sweeps by one thread
    [2, 3, 50, 51, 52, 400, 2000, 2001, 2002, 2003, 5000],   # spacings that jump by three orders of magnitude
])
def test_spline_kernel_on_smooth_spectra_against_the_oracle(los, l_list):
    l_list = np.asarray(l_list, dtype=np.int32)
    l = l_list.astype(np.float64)
    # smooth positive TT, EE and a sign-changing TE with acoustic-like wiggles, shaped like CMB spectra
    tt = (1.0 + 0.5 * np.cos(l / 70.0)) * np.exp(-(l / 1400.0) ** 1.2) / (l * (l + 1.0))
    ee = 0.02 * (1.0 + 0.7 * np.sin(l / 70.0)) * np.exp(-(l / 1800.0) ** 1.2) / (l * (l + 1.0))
    te = 0.1 * np.sin(l / 35.0) * np.sqrt(tt * ee)
    C = np.stack([tt, ee, te])
    plan = small_plan(los, l_list)
    out = plan.gcamb_los_cl_interp(dev(C))
    torch.cuda.synchronize()
    ref = oracle.cl_interp(l_list, C, real="f80")
    assert out.shape == ref.shape == (3, l_list[-1] - l_list[0] + 1)
    # Across a long gap the spline of a wiggly spectrum swings through zero, so the error is measured in
    # the interpolated quantity y = l (l+1) C_l against the largest |y| of the series
    l_all = np.arange(l_list[0], l_list[-1] + 1, dtype=np.float64)
    y_gpu, y_ref = out.cpu().numpy() * l_all * (l_all + 1.0), ref * l_all * (l_all + 1.0)
    err = np.max(np.abs(y_gpu - y_ref), axis=-1) / np.max(np.abs(y_ref), axis=-1)
    assert np.all(err <= 1e-12), err
    # the listed multipoles come back unchanged (up to the rounding of y / (l (l+1)))
    assert np.max(np.abs(out.cpu().numpy()[:, l_list - l_list[0]] / C - 1.0)) <= 4e-16
    # deterministic
    assert torch.equal(out, plan.gcamb_los_cl_interp(dev(C)))
    plan.close()


def test_batched_interp_equals_a_loop_of_single_calls_and_handles_phi(los):
    l_list = camb_like_list(2, 900, dense_to=20, step_mid=7, mid_to=150, step_hi=37)
    rng = np.random.default_rng(7)
    k = np.geomspace(1e-4, 0.1, 8)
    tau = np.linspace(100.0, 13000.0, 40)
    plan = los.Plan(l_list, k, tau, 14000.0, with_phi=True)
    l = l_list.astype(np.float64)
    C = rng.uniform(0.5, 1.5, size=(5, 4, l_list.size)) / (l * (l + 1.0))
    out = plan.gcamb_los_cl_interp(dev(C))
    assert out.shape == (5, 4, 899)
    for b in range(5):
        assert torch.equal(out[b], plan.gcamb_los_cl_interp(dev(C[b])))
        ref = oracle.cl_interp(l_list, C[b], real="f80")
        l_all = np.arange(2, 901, dtype=np.float64)
        dy = (out[b].cpu().numpy() - ref) * l_all * (l_all + 1.0)          # y is O(1) here
        assert np.max(np.abs(dy)) <= 1e-12
    plan.close()


def test_config1_sparse_l_pipeline_against_the_oracle(los):
    """Config-1 grids, CAMB-like list of 101 multipoles (every l below 40, every 10th to 200, every 50th
    above): transfer -> cls -> interp on the GPU against the same steps of the long-double oracle."""
    cfg = synth.CONFIGS[1]
    l_sparse = camb_like_list(cfg.l_min, cfg.l_max)
    S_T, S_E, _ = synth.sources(cfg)
    P = synth.primordial_power(cfg)
    plan = los.Plan(l_sparse, cfg.k(), cfg.tau(), cfg.tau0)
    D = plan.gcamb_los_transfer(dev(S_T), dev(S_E))
    C = plan.gcamb_los_cls(D, dev(P))
    C_all = torch.full((3, cfg.n_l), float("nan"), dtype=torch.float64, device="cuda")
    plan.gcamb_los_cl_interp(C, out=C_all)
    torch.cuda.synchronize()
    D_ref = oracle.transfer(l_sparse, cfg.k(), cfg.tau(), cfg.tau0, S_T, S_E, real="f80")
    C_ref = oracle.cls(cfg.k(), D_ref, P, real="f80")
    ref = oracle.cl_interp(l_sparse, C_ref, real="f80")
    got = C_all.cpu().numpy()
    assert np.all(np.isfinite(got))
    e_auto, e_te = interp_err(got, ref)
    assert e_auto <= TOL_CL and e_te <= TOL_CL, (e_auto, e_te)
    plan.close()


def test_interp_error_paths(los):
    plan = small_plan(los, np.array([7], dtype=np.int32))          # one multipole: nothing to interpolate
    with pytest.raises(los.GcambError) as e:
        plan.gcamb_los_cl_interp(torch.zeros(3, 1, dtype=torch.float64, device="cuda"))
    assert e.value.status == 1
    plan.close()
    plan = small_plan(los, np.arange(2, 10003, dtype=np.int32))    # 10001 knots > 10000
    with pytest.raises(los.GcambError) as e:
        plan.gcamb_los_cl_interp(torch.zeros(3, 10001, dtype=torch.float64, device="cuda"))
    assert e.value.status == 1 and "10000" in str(e.value)
    plan.close()
