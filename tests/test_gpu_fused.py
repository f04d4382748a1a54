"""gcamb_los_spectra_batched: sources of a batch -> C_l in one fused kernel that shares the j_l
recurrence across the cosmologies of a block and never writes Delta (emulator
use-case PAPER.md:24, 248).  Checked against the long-double oracle (C_l to 1e-8, reading R13),
against the two-kernel GPU path (same sums in another order: agreement far inside the bar), for
run-to-run bit equality, for ragged batches, and for the plans that fall back to the two kernels.
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


def cl_err(C_gpu, C_ref):
    auto = [0, 1] + ([3] if C_ref.shape[-2] == 4 else [])
    e_auto = float(np.max(np.abs(C_gpu[..., auto, :] / C_ref[..., auto, :] - 1.0)))
    norm = np.sqrt(C_ref[..., 2, :] ** 2 + C_ref[..., 0, :] * C_ref[..., 1, :])
    e_te = float(np.max(np.abs(C_gpu[..., 2, :] - C_ref[..., 2, :]) / norm))
    return e_auto, e_te


def batch_inputs(cfg):
    S = [synth.sources(cfg, c) for c in range(cfg.n_batch)]
    hS = [np.stack([s[q] for s in S]) if S[0][q] is not None else None for q in range(3)]
    hP = np.stack([synth.primordial_power(cfg, c) for c in range(cfg.n_batch)])
    return hS, hP


@pytest.mark.parametrize("shape", [
    # (l_max, n_k, n_tau_uniform, n_tau_log, batch): block of 8 with T = 1..5, ragged batches, block of 4
    (300, 40, 120, 60, 8),
    (200, 37, 200, 100, 5),
    (420, 25, 400, 241, 11),
    (150, 18, 600, 600, 16),
    (260, 30, 100, 29, 3),
    (180, 12, 900, 700, 4),       # n_tau = 1600 > 1280: blocks of 4 cosmologies
    (90, 9, 1300, 1260, 9),       # n_tau = 2560: the largest grid the fused kernel holds
])
def test_fused_matches_oracle_and_two_kernel_path(los, shape):
    l_max, n_k, n_u, n_log, B = shape
    cfg = synth.Config(9, "fused", 2, l_max, n_k, 1e-4, 0.3, n_u, n_log, False, n_batch=B)
    hS, hP = batch_inputs(cfg)
    plan = los.Plan(cfg.l_list(), cfg.k(), cfg.tau(), cfg.tau0)
    info = plan.gcamb_los_spectra_batched_info(B)
    assert info["fused"] and info["kernels"] == 2
    d_T, d_E, d_P = dev(hS[0]), dev(hS[1]), dev(hP)
    C = torch.full((B, 3, cfg.n_l), float("nan"), dtype=torch.float64, device="cuda")
    plan.gcamb_los_spectra_batched(d_T, d_E, None, d_P, out=C)
    C2 = torch.full_like(C, float("nan"))
    plan.gcamb_los_spectra_batched(d_T, d_E, None, d_P, out=C2)
    torch.cuda.synchronize()
    assert torch.equal(C, C2)                         # fixed summation order: bit-reproducible
    C_two = plan.gcamb_los_cls_batched(plan.gcamb_los_transfer_batched(d_T, d_E), d_P).cpu().numpy()
    C = C.cpu().numpy()
    assert np.all(np.isfinite(C))
    e_auto, e_te = cl_err(C, C_two)
    assert e_auto <= 1e-11 and e_te <= 1e-11, (e_auto, e_te)
    for c in range(B):
        D_ref = oracle.transfer(cfg.l_list(), cfg.k(), cfg.tau(), cfg.tau0, hS[0][c], hS[1][c], real="f80")
        C_ref = oracle.cls(cfg.k(), D_ref, hP[c], real="f80")
        e_auto, e_te = cl_err(C[c], C_ref)
        assert e_auto <= TOL_CL and e_te <= TOL_CL, (c, e_auto, e_te)
    plan.close()


def test_fused_does_not_depend_on_the_other_cosmologies(los):
    """A cosmology's spectra must not change with what else is in its block or in the batch."""
    cfg = synth.Config(9, "fused", 2, 200, 33, 1e-4, 0.3, 150, 80, False, n_batch=10)
    hS, hP = batch_inputs(cfg)
    plan = los.Plan(cfg.l_list(), cfg.k(), cfg.tau(), cfg.tau0)
    C_all = plan.gcamb_los_spectra_batched(dev(hS[0]), dev(hS[1]), None, dev(hP))
    sel = [8, 9, 0, 1, 2, 3, 4]           # other block composition, other positions
    C_sel = plan.gcamb_los_spectra_batched(dev(hS[0][sel]), dev(hS[1][sel]), None, dev(hP[sel]))
    torch.cuda.synchronize()
    assert torch.equal(C_sel, C_all[sel])
    plan.close()


def test_fused_with_a_sparse_l_list(los):
    """CAMB's default operating mode (`l_sample_boost`): only the listed l are accumulated."""
    cfg = synth.Config(9, "fused-sparse", 2, 700, 30, 1e-4, 0.3, 150, 80, False, n_batch=6)
    l_list = np.unique(np.concatenate([np.arange(2, 20), np.arange(20, 100, 10), np.arange(100, 701, 50)])).astype(np.int32)
    hS, hP = batch_inputs(cfg)
    plan = los.Plan(l_list, cfg.k(), cfg.tau(), cfg.tau0)
    assert plan.gcamb_los_spectra_batched_info(6)["fused"]
    C = plan.gcamb_los_spectra_batched(dev(hS[0]), dev(hS[1]), None, dev(hP)).cpu().numpy()
    for c in (0, 5):
        D_ref = oracle.transfer(l_list, cfg.k(), cfg.tau(), cfg.tau0, hS[0][c], hS[1][c], real="f80")
        C_ref = oracle.cls(cfg.k(), D_ref, hP[c], real="f80")
        e_auto, e_te = cl_err(C[c], C_ref)
        assert e_auto <= TOL_CL and e_te <= TOL_CL
    plan.close()


@pytest.mark.parametrize("shape", [
    # (l_max, n_k, n_tau_uniform, n_tau_log, batch): the recurrence-only tiles with 1..10 slots per thread
    (900, 20, 600, 600, 8),        # T = 5, blocks of 8 cosmologies
    (700, 14, 250, 133, 9),        # T = 2, ragged batch, odd n_tau
    (600, 10, 900, 700, 5),        # n_tau = 1600 > 1280: blocks of 4, T = 8
    (500, 8, 1300, 1260, 4),       # n_tau = 2560: T = 10
])
def test_fused_sparse_lists_against_the_two_kernel_path_and_the_oracle(los, shape):
    l_max, n_k, n_u, n_log, B = shape
    cfg = synth.Config(9, "fused-sparse-shapes", 2, l_max, n_k, 1e-4, 0.3, n_u, n_log, False, n_batch=B)
    rng = np.random.default_rng(l_max)
    l_list = np.unique(np.concatenate([np.arange(2, 12), rng.choice(np.arange(12, l_max), size=25, replace=False),
                                       [l_max]])).astype(np.int32)
    hS, hP = batch_inputs(cfg)
    plan = los.Plan(l_list, cfg.k(), cfg.tau(), cfg.tau0)
    assert plan.gcamb_los_spectra_batched_info(B)["fused"]
    d_T, d_E, d_P = dev(hS[0]), dev(hS[1]), dev(hP)
    C = torch.full((B, 3, l_list.size), float("nan"), dtype=torch.float64, device="cuda")
    plan.gcamb_los_spectra_batched(d_T, d_E, None, d_P, out=C)
    torch.cuda.synchronize()
    assert torch.equal(C, plan.gcamb_los_spectra_batched(d_T, d_E, None, d_P))        # deterministic
    C_two = plan.gcamb_los_cls_batched(plan.gcamb_los_transfer_batched(d_T, d_E), d_P).cpu().numpy()
    C = C.cpu().numpy()
    assert np.all(np.isfinite(C))
    e_auto, e_te = cl_err(C, C_two)                                                    # same sums in another order
    assert e_auto <= 1e-11 and e_te <= 1e-11
    c = B - 1
    D_ref = oracle.transfer(l_list, cfg.k(), cfg.tau(), cfg.tau0, hS[0][c], hS[1][c], real="f80")
    e_auto, e_te = cl_err(C[c], oracle.cls(cfg.k(), D_ref, hP[c], real="f80"))
    assert e_auto <= TOL_CL and e_te <= TOL_CL
    plan.close()


def test_emulator_step_captures_into_a_cuda_graph(los):
    """SURVEY 8(f) NEXT-1, second half: the whole batched step (fused kernel, finish kernel, spline to every l)
    only enqueues work on the caller's stream, so an emulator loop captures it once and replays it on new
    sources written into the same buffers."""
    cfg = synth.Config(9, "fused-graph", 2, 700, 30, 1e-4, 0.3, 150, 80, False, n_batch=8)
    l_list = np.unique(np.concatenate([np.arange(2, 20), np.arange(20, 100, 10), np.arange(100, 701, 50)])).astype(np.int32)
    hS, hP = batch_inputs(cfg)
    plan = los.Plan(l_list, cfg.k(), cfg.tau(), cfg.tau0)
    assert plan.gcamb_los_spectra_batched_info(8)["fused"]
    d_T, d_E, d_P = dev(hS[0]), dev(hS[1]), dev(hP)
    C = torch.empty(8, 3, l_list.size, dtype=torch.float64, device="cuda")
    C_all = torch.empty(8, 3, 699, dtype=torch.float64, device="cuda")
    plan.gcamb_los_spectra_batched(d_T, d_E, None, d_P, out=C)           # first call: one-time function attributes
    plan.gcamb_los_cl_interp(C, out=C_all)
    torch.cuda.synchronize()
    C0, C_all0 = C.clone(), C_all.clone()
    graph, side = torch.cuda.CUDAGraph(), torch.cuda.Stream()
    with torch.cuda.stream(side):
        with torch.cuda.graph(graph, stream=side):
            plan.gcamb_los_spectra_batched(d_T, d_E, None, d_P, out=C)
            plan.gcamb_los_cl_interp(C, out=C_all)
    for _ in range(2):
        C.fill_(float("nan"))
        C_all.fill_(float("nan"))
        graph.replay()
        torch.cuda.synchronize()
        assert torch.equal(C, C0) and torch.equal(C_all, C_all0)
    # new cosmologies in the same buffers: the replay computes what a direct call computes
    perm = torch.tensor([3, 0, 7, 1, 6, 2, 5, 4], device="cuda")
    d_T.copy_(d_T[perm].clone()); d_E.copy_(d_E[perm].clone()); d_P.copy_(d_P[perm].clone())
    graph.replay()
    torch.cuda.synchronize()
    assert torch.equal(C, C0[perm]) and torch.equal(C_all, C_all0[perm])
    plan.close()


@pytest.mark.parametrize("case", ["phi", "single", "long_tau"])
def test_plans_outside_the_fused_kernel_take_the_two_kernel_path(los, case):
    with_phi = case == "phi"
    B = 1 if case == "single" else 4
    n_u, n_log = (1500, 1200) if case == "long_tau" else (100, 60)
    cfg = synth.Config(9, "fallback", 2, 120, 20, 1e-4, 0.2, n_u, n_log, with_phi, n_batch=B)
    l_list = cfg.l_list()
    hS, hP = batch_inputs(cfg)
    plan = los.Plan(l_list, cfg.k(), cfg.tau(), cfg.tau0, with_phi=with_phi)
    info = plan.gcamb_los_spectra_batched_info(B)
    assert not info["fused"] and info["scratch_bytes"] == 8 * B * plan.n_src * plan.n_l * plan.n_k
    d = [None if x is None else dev(x) for x in hS]
    C = plan.gcamb_los_spectra_batched(d[0], d[1], d[2], dev(hP))
    C_two = plan.gcamb_los_cls_batched(plan.gcamb_los_transfer_batched(d[0], d[1], d[2]), dev(hP))
    torch.cuda.synchronize()
    assert torch.equal(C, C_two)
    plan.close()


def test_config3_fused_against_the_oracle(los):
    """BASELINE.json config 3 at full size through the fused kernel: 64 cosmologies, one call; eight
    of them compared with the long-double oracle, all 64 with the two-kernel path."""
    cfg = synth.CONFIGS[3]
    B = cfg.n_batch
    plan = los.Plan(cfg.l_list(), cfg.k(), cfg.tau(), cfg.tau0)
    S_T = torch.empty(B, cfg.n_k, cfg.n_tau, dtype=torch.float64, device="cuda")
    S_E = torch.empty_like(S_T)
    P = torch.empty(B, cfg.n_k, dtype=torch.float64, device="cuda")
    check = tuple(range(3, 64, 8))
    host = {}
    for c in range(B):
        s = synth.sources(cfg, c)
        S_T[c].copy_(torch.from_numpy(s[0]))
        S_E[c].copy_(torch.from_numpy(s[1]))
        pr = synth.primordial_power(cfg, c)
        P[c].copy_(torch.from_numpy(pr))
        if c in check:
            host[c] = (s, pr)
    assert plan.gcamb_los_spectra_batched_info(B)["fused"]
    C = torch.full((B, 3, cfg.n_l), float("nan"), dtype=torch.float64, device="cuda")
    plan.gcamb_los_spectra_batched(S_T, S_E, None, P, out=C)
    C2 = plan.gcamb_los_spectra_batched(S_T, S_E, None, P)
    torch.cuda.synchronize()
    assert torch.equal(C, C2)
    C_two = plan.gcamb_los_cls_batched(plan.gcamb_los_transfer_batched(S_T, S_E), P).cpu().numpy()
    C = C.cpu().numpy()
    e_auto, e_te = cl_err(C, C_two)
    assert e_auto <= 1e-10 and e_te <= 1e-10, (e_auto, e_te)
    for c in check:
        s, pr = host[c]
        D_ref = oracle.transfer(cfg.l_list(), cfg.k(), cfg.tau(), cfg.tau0, s[0], s[1], real="f80")
        C_ref = oracle.cls(cfg.k(), D_ref, pr, real="f80")
        e_auto, e_te = cl_err(C[c], C_ref)
        assert e_auto <= TOL_CL and e_te <= TOL_CL, (c, e_auto, e_te)
    plan.close()
