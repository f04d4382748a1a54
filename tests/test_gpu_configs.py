"""GPU parity at BASELINE.json's full config sizes, in the launch configuration bench.py times.

Configs 1 and 2 are compared element by element with the long-double oracle (the whole Delta
and C_l).  Config 3 runs all 64 cosmologies in one batched launch pair and compares sixteen of
them in full.  Config 4 (4.8 GB of Delta) is compared with the oracle on EVERY k row, in ten
sub-problems of every 10th k (offsets 0..9; same l range, same tau grid, hence the same CTA shape
and the same per-k work):
  * the full-size run is checked on properties (every element written and finite, zero exactly
    where R16 says so, TT/EE/phiphi >= 0, Cauchy-Schwarz for TE),
  * each sub-problem's rows must equal the full run's rows bit for bit (a k row never depends on
    the other rows) and are compared element by element with the long-double oracle; the per-l
    error is then formed over all 20000 k rows (largest |difference| over all rows / largest
    |Delta_l| over all rows), and the first sub-problem's C_l is compared too.
Outputs are pre-filled with NaN so an element the kernels fail to write cannot pass.

Bars as in test_gpu_parity.py: |dDelta| <= 1e-10 max_k|Delta_l| per (source, l); C_l 1e-8 (R13).

Config 4, l > ~8500, sources T and E (reading R14): there the synthetic
recombination signal is damped to 1e-26 ... 1e-32 and the tau-sum cancels down to the +-1e-3 noise, so
that ANY fp64 evaluation loses five digits: over all 20000 k rows the fp64 build of the oracle differs
from the long-double build by up to 4.0e-11 max_k|Delta_l|, the GPU path by up to 3.2e-11.  With the
normaliser BASELINE.json states (the largest |Delta_l| over ALL k of the config) both are inside the plain
1e-10, and that is what the test asserts: no allowance.  (On a subset of the k rows the normaliser is
smaller: on every 10th row alone the same differences read 1.2e-10, which is why round 1, which compared
that subset only, carried an allowance.)  The fp64 oracle is run on every k row as well and printed beside
the GPU figure; DESIGN.md 6.3 carries both, and those of the one variant tried against the floor
(coefficient carried as hi + lo through the recurrence step: no gain, +27 % time).
"""
import numpy as np
import pytest
import torch

import oracle
from paper_2509_25110_b200 import synth

pytestmark = pytest.mark.gpu

TOL_DELTA = 1e-10
TOL_CL = 1e-8


@pytest.fixture(scope="module")
def los():
    from paper_2509_25110_b200 import los as _los
    _los.load_library()
    assert torch.cuda.is_available()
    return _los


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def nan_like(*shape):
    return torch.full(shape, float("nan"), dtype=torch.float64, device="cuda")


def delta_err(D_gpu, D_ref):
    """per (source, l): max_k |diff| / max_k |Delta_l|; returns the worst ratio and where."""
    scale = np.max(np.abs(D_ref), axis=-1)
    err = np.max(np.abs(D_gpu - D_ref), axis=-1)
    ratio = err / np.where(scale > 0, scale, 1.0)
    q, a = np.unravel_index(np.argmax(ratio), ratio.shape)
    return float(ratio[q, a]), (int(q), int(a))


def cl_err(C_gpu, C_ref):
    auto = [0, 1] + ([3] if C_ref.shape[-2] == 4 else [])
    e_auto = float(np.max(np.abs(C_gpu[..., auto, :] / C_ref[..., auto, :] - 1.0)))
    norm = np.sqrt(C_ref[..., 2, :] ** 2 + C_ref[..., 0, :] * C_ref[..., 1, :])
    e_te = float(np.max(np.abs(C_gpu[..., 2, :] - C_ref[..., 2, :]) / norm))
    return e_auto, e_te


def cl_properties(C):
    auto = [0, 1] + ([3] if C.shape[-2] == 4 else [])
    assert np.all(np.isfinite(C))
    assert np.all(C[..., auto, :] >= 0.0)
    # Cauchy-Schwarz holds exactly for positive weights; allow rounding of the three sums
    assert np.all(C[..., 2, :] ** 2 <= C[..., 0, :] * C[..., 1, :] * (1 + 1e-12))


def run_single(los, cfg, k_slice=slice(None)):
    k = cfg.k()[k_slice]
    S_T, S_E, S_P = synth.sources(cfg, 0, k_slice)
    P = synth.primordial_power(cfg, 0)[k_slice]
    plan = los.Plan(cfg.l_list(), k, cfg.tau(), cfg.tau0, with_phi=cfg.with_phi)
    D = nan_like(plan.n_src, plan.n_l, plan.n_k)
    C = nan_like(plan.n_spec, plan.n_l)
    plan.gcamb_los_transfer(dev(S_T), dev(S_E), None if S_P is None else dev(S_P), out=D)
    plan.gcamb_los_cls(D, dev(P), out=C)
    torch.cuda.synchronize()
    return plan, k, (S_T, S_E, S_P), P, D, C


def oracle_run(cfg, k, S, P):
    D_ref = oracle.transfer(cfg.l_list(), k, cfg.tau(), cfg.tau0, S[0], S[1], S[2], real="f80")
    C_ref = oracle.cls(k, D_ref, P, real="f80")
    return D_ref, C_ref


@pytest.mark.parametrize("index", [1, 2])
def test_full_config_element_by_element(los, index):
    cfg = synth.CONFIGS[index]
    plan, k, S, P, D, C = run_single(los, cfg)
    assert plan.nominal_terms == cfg.nominal_terms()
    D, C = D.cpu().numpy(), C.cpu().numpy()
    assert np.all(np.isfinite(D))
    cl_properties(C)
    D_ref, C_ref = oracle_run(cfg, k, S, P)
    e, where = delta_err(D, D_ref)
    assert e <= TOL_DELTA, f"config {index}: Delta error {e:.3e} at (source, l index) {where}"
    e_auto, e_te = cl_err(C, C_ref)
    assert e_auto <= TOL_CL and e_te <= TOL_CL
    # R16: exact zeros of the oracle (l above the cut of every tau) are exact zeros on the GPU
    assert np.all(D[D_ref == 0.0] == 0.0)
    plan.close()


def test_config3_emulator_batch(los):
    cfg = synth.CONFIGS[3]
    B = cfg.n_batch
    plan = los.Plan(cfg.l_list(), cfg.k(), cfg.tau(), cfg.tau0)
    S_T = torch.empty(B, cfg.n_k, cfg.n_tau, dtype=torch.float64, device="cuda")
    S_E = torch.empty_like(S_T)
    P = torch.empty(B, cfg.n_k, dtype=torch.float64, device="cuda")
    host = {}
    check = tuple(range(0, 64, 4))          # 16 of the 64 cosmologies, element by element
    for c in range(B):
        s = synth.sources(cfg, c)
        S_T[c].copy_(torch.from_numpy(s[0]))
        S_E[c].copy_(torch.from_numpy(s[1]))
        pr = synth.primordial_power(cfg, c)
        P[c].copy_(torch.from_numpy(pr))
        if c in check:
            host[c] = (s, pr)
    D = nan_like(B, plan.n_src, plan.n_l, plan.n_k)
    C = nan_like(B, plan.n_spec, plan.n_l)
    plan.gcamb_los_transfer_batched(S_T, S_E, out=D)
    plan.gcamb_los_cls_batched(D, P, out=C)
    torch.cuda.synchronize()
    assert bool(torch.isfinite(D).all())
    C_h = C.cpu().numpy()
    cl_properties(C_h)
    for c in check:
        s, pr = host[c]
        D_ref, C_ref = oracle_run(cfg, cfg.k(), s, pr)
        e, where = delta_err(D[c].cpu().numpy(), D_ref)
        assert e <= TOL_DELTA, f"cosmology {c}: Delta error {e:.3e} at {where}"
        e_auto, e_te = cl_err(C_h[c], C_ref)
        assert e_auto <= TOL_CL and e_te <= TOL_CL
    # the batched launch equals the single-cosmology launch bit for bit
    D1 = plan.gcamb_los_transfer(S_T[5].contiguous(), S_E[5].contiguous())
    assert torch.equal(D1, D[5])
    plan.close()


def test_config4_extreme(los):
    cfg = synth.CONFIGS[4]
    stride = 10
    plan, k, S, P, D, C = run_single(los, cfg)
    assert plan.nominal_terms == cfg.nominal_terms()
    assert bool(torch.isfinite(D).all())
    cl_properties(C.cpu().numpy())
    del C, S
    plan.close()

    n_src, n_l = 3, cfg.n_l
    err = np.zeros((n_src, n_l)); err64 = np.zeros((n_src, n_l)); scale = np.zeros((n_src, n_l))
    for off in range(stride):
        sl = slice(off, cfg.n_k, stride)
        rows = torch.arange(off, cfg.n_k, stride, device="cuda")
        plan_s, k_s, S_s, P_s, D_s, C_s = run_single(los, cfg, sl)
        assert torch.equal(D_s, D[:, :, rows])          # a k row does not depend on the other rows
        D_s = D_s.cpu().numpy()
        D_ref, C_ref = oracle_run(cfg, k_s, S_s, P_s)
        D_f64 = oracle.transfer(cfg.l_list(), k_s, cfg.tau(), cfg.tau0, S_s[0], S_s[1], S_s[2], real="f64")
        err = np.maximum(err, np.max(np.abs(D_s - D_ref), axis=-1))
        err64 = np.maximum(err64, np.max(np.abs(D_f64 - D_ref), axis=-1))
        scale = np.maximum(scale, np.max(np.abs(D_ref), axis=-1))
        assert np.all(D_s[D_ref == 0.0] == 0.0)
        if off == 0:
            e_auto, e_te = cl_err(C_s.cpu().numpy(), C_ref)
            assert e_auto <= TOL_CL and e_te <= TOL_CL
        plan_s.close()
        del D_s, D_ref, D_f64, S_s
    scale = np.where(scale > 0, scale, 1.0)
    e_gpu = err / scale            # [source][l], over all 20000 k rows
    e_f64 = err64 / scale          # the fp64 floor, same rows, same normaliser
    over = e_gpu > TOL_DELTA
    print(f"config 4, all {cfg.n_k} k rows: max Delta error {e_gpu.max():.3e}; l over 1e-10 per source: "
          f"{over.sum(axis=1).tolist()}; fp64 oracle vs long double: max {e_f64.max():.3e}, "
          f"l over 1e-10: {(e_f64 > TOL_DELTA).sum(axis=1).tolist()}")
    assert np.all(e_gpu <= TOL_DELTA), "Delta error above 1e-10 max_k|Delta_l|"      # the plain bar of BASELINE.json
    assert e_gpu.max() <= 1.5 * e_f64.max()                       # and no worse than the fp64 floor of the method
    assert np.all(e_gpu[2] <= 0.01 * TOL_DELTA)                   # the lensing source is far from that regime
    # below l = 7000 the plain bar holds with margin
    assert np.all(e_gpu[:, : 7000 - cfg.l_min] <= 0.2 * TOL_DELTA)


def test_config1_sparse_l_list_equals_the_dense_rows(los):
    """R21 at config-1 size: an l list sampled like CAMB's default (every l at low l, every 50th
    above; `l_sample_boost`).  Tiles without a listed l are walked by the
    recurrence only; the listed rows must equal those of the all-l run bit for bit."""
    cfg = synth.CONFIGS[1]
    l_sparse = np.unique(np.concatenate([np.arange(2, 40), np.arange(40, 200, 10),
                                         np.arange(200, 2501, 50), [2499, 2500]])).astype(np.int32)
    S_T, S_E, _ = synth.sources(cfg)
    d_T, d_E = dev(S_T), dev(S_E)
    dense = los.Plan(cfg.l_list(), cfg.k(), cfg.tau(), cfg.tau0)
    sparse = los.Plan(l_sparse, cfg.k(), cfg.tau(), cfg.tau0)
    D_dense = dense.gcamb_los_transfer(d_T, d_E)
    D_sparse = nan_like(2, l_sparse.size, cfg.n_k)
    sparse.gcamb_los_transfer(d_T, d_E, out=D_sparse)
    torch.cuda.synchronize()
    rows = torch.from_numpy(l_sparse.astype(np.int64) - cfg.l_min).cuda()
    assert torch.equal(D_sparse, D_dense[:, rows, :])
    dense.close()
    sparse.close()
