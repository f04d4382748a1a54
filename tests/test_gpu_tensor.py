"""SURVEY 8(f) NEXT-3 on the GPU: tensor-mode transfer functions and spectra (reading R27) and the
interpolation of the sources in k (reading R26, `InterpolateSources`), element by element
against the long-double oracle (pinned in tests/test_oracle_tensor.py).

Bars as for the scalars (BASELINE.json north_star): |dDelta| <= 1e-10 max_k|Delta_l| per (source, l);
C_l relative 1e-8 for the auto spectra TT, EE, BB, and for TE relative to sqrt(TE^2 + TT EE) (R13).

Inputs: seeded synthetic tensor sources shaped like the scalar ones of BASELINE.json (visibility peak at
recombination, damping in k, +-1e-3 relative noise from the same counter-based generator), on the tensor
grid sizes the paper quotes: l_max_tensor = 1500, k tau0 up to 3000.
"""
import numpy as np
import pytest
import torch

import oracle
from paper_2509_25110_b200 import synth

pytestmark = pytest.mark.gpu

TOL_DELTA = 1e-10
TOL_CL = 1e-8
TAU0 = 14000.0


@pytest.fixture(scope="module")
def los():
    from paper_2509_25110_b200 import los as _los
    _los.load_library()
    assert torch.cuda.is_available()
    return _los


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def tensor_sources(k, tau, seed=1234):
    """S_T, S_E, S_B of the tensor modes [n_k][n_tau]: a visibility peak at recombination times a damped
    oscillation in k tau (gravitational-wave like), a late-time term in S_T, seeded +-1e-3 noise."""
    kk, tt = k[:, None], tau[None, :]
    g = np.exp(-((tt - 280.0) ** 2) / (2.0 * 20.0 ** 2)) / (20.0 * np.sqrt(2.0 * np.pi))
    damp = np.exp(-((kk / 0.05) ** 2))
    h = np.sin(kk * tt) / (kk * tt)                       # the tensor mode function of a radiation universe
    S_T = g * h * damp + 0.3 * np.exp(-(((tt - 10000.0) / 2500.0) ** 2)) * np.exp(-kk / 0.005) * 1e-4
    S_E = g * h * damp * 0.2
    S_B = g * np.cos(kk * tt) * damp * 0.15
    out = []
    for q, S in enumerate((S_T, S_E, S_B)):
        u = synth.uniform_pm1(seed, 500 + q, 0, k.size * tau.size).reshape(k.size, tau.size)
        out.append(np.ascontiguousarray(S * (1.0 + 1e-3 * u)))
    return out


def delta_err(D_gpu, D_ref):
    scale = np.max(np.abs(D_ref), axis=-1)
    err = np.max(np.abs(D_gpu - D_ref), axis=-1)
    return err / np.where(scale > 0, scale, 1.0)


def cl_err(C, C_ref):
    e_auto = float(np.max(np.abs(C[:3] / C_ref[:3] - 1.0)))
    e_te = float(np.max(np.abs(C[3] - C_ref[3]) / np.sqrt(C_ref[3] ** 2 + C_ref[0] * C_ref[1])))
    return e_auto, e_te


def run_tensor(los, l_list, k, tau, S, P_t):
    plan = los.Plan(l_list, k, tau, TAU0, tensor=True)
    assert (plan.n_l, plan.n_src, plan.n_spec) == (len(l_list), 3, 4)
    D = torch.full((3, plan.n_l, plan.n_k), float("nan"), dtype=torch.float64, device="cuda")
    C = torch.full((4, plan.n_l), float("nan"), dtype=torch.float64, device="cuda")
    d_S = [dev(s) for s in S]
    plan.gcamb_los_transfer_tensor(*d_S, out=D)
    plan.gcamb_los_cls_tensor(D, dev(P_t), out=C)
    torch.cuda.synchronize()
    D2 = plan.gcamb_los_transfer_tensor(*d_S)                  # deterministic
    assert torch.equal(D, D2)
    return plan, D.cpu().numpy(), C.cpu().numpy()


@pytest.mark.parametrize("case", [
    dict(l=np.arange(2, 201), n_k=60, k_hi=0.02, n_u=120, n_log=60),
    dict(l=np.arange(2, 90), n_k=33, k_hi=0.3, n_u=40, n_log=29),            # x far above l_max: every point starts at the top
    dict(l=np.array([2, 3, 4, 9, 10, 30, 31, 32, 77, 150, 151, 400]), n_k=41, k_hi=0.05, n_u=200, n_log=100),   # sparse list: l and l+1 overlap
    dict(l=np.array([65533]), n_k=5, k_hi=0.01, n_u=20, n_log=12),           # largest tensor multipole; nothing reaches it
])
def test_tensor_small_shapes_against_the_oracle(los, case):
    l_list = case["l"].astype(np.int32)
    k = synth.k_grid(case["n_k"], 1e-4, case["k_hi"])
    tau = synth.tau_grid(case["n_u"], case["n_log"], TAU0)
    S = tensor_sources(k, tau)
    P_t = 2.1e-10 * (k / 0.05) ** -0.01
    plan, D, C = run_tensor(los, l_list, k, tau, S, P_t)
    assert np.all(np.isfinite(D)) and np.all(np.isfinite(C))
    D_ref = oracle.transfer_tensor(l_list, k, tau, TAU0, *S, real="f80")
    e = delta_err(D, D_ref)
    assert np.all(e <= TOL_DELTA), (float(e.max()), np.unravel_index(np.argmax(e), e.shape))
    if np.all(np.max(np.abs(D_ref), axis=-1) > 0):
        C_ref = oracle.cls_tensor(k, D_ref, P_t, real="f80")
        e_auto, e_te = cl_err(C, C_ref)
        assert e_auto <= TOL_CL and e_te <= TOL_CL
        # the C_l kernels alone on the oracle's transfer functions: rounding level, order TT, EE, BB, TE
        C2 = plan.gcamb_los_cls_tensor(dev(D_ref), dev(P_t)).cpu().numpy()
        e_auto, e_te = cl_err(C2, C_ref)
        assert e_auto <= 1e-13 and e_te <= 1e-13
    else:
        assert np.all(D == 0.0) and np.all(C == 0.0)
    plan.close()


@pytest.mark.parametrize("case", [
    dict(n_k=24, n_u=1000, n_log=700),    # 1700 tau: one pass of 256 threads x 7 points
    dict(n_k=16, n_u=2000, n_log=1300),   # 3300 tau: two passes of 128 threads x 12 points
])
def test_tensor_four_sum_kernels_on_compensated_rows_and_tau_passes(los, case):
    """The other instantiations of the four-sum transfer kernels: k tau0 up to 12600 > 6755, so the largest k run the
    compensated coefficient in a launch of their own, and tau grids beyond 128 x 12 points."""
    l_list = np.arange(2, 301, dtype=np.int32)
    k = synth.k_grid(case["n_k"], 1e-3, 0.9)
    tau = synth.tau_grid(case["n_u"], case["n_log"], TAU0)
    n_comp = int(np.sum(k * TAU0 > 6755.4))
    assert 2 <= n_comp < k.size
    # sources in phase with j_l(k (tau0 - tau)) (no cancellation in the tau-sum) and without the damping in k of
    # tensor_sources, so that the rows of the largest k carry signal
    kk, tt = k[:, None], tau[None, :]
    S = []
    for q, (amp, ph) in enumerate(((1.0, 0.4), (0.2, 1.1), (0.15, 2.3))):
        u = synth.uniform_pm1(1234, 520 + q, 0, k.size * tau.size).reshape(k.size, tau.size)
        S.append(np.ascontiguousarray(amp * 1e-4 * np.cos(kk * (TAU0 - tt) + ph) * (1.0 + 1e-3 * u)))
    P_t = 2.1e-10 * (k / 0.05) ** -0.01
    plan, D, C = run_tensor(los, l_list, k, tau, S, P_t)
    assert np.all(np.isfinite(D)) and np.all(np.isfinite(C))
    D_ref = oracle.transfer_tensor(l_list, k, tau, TAU0, *S, real="f80")
    # the compensated rows are not negligible next to the others
    assert np.all(np.max(np.abs(D_ref[:, :, -n_comp:]), axis=(1, 2)) >= 1e-3 * np.max(np.abs(D_ref), axis=(1, 2)))
    e = delta_err(D, D_ref)
    assert np.all(e <= TOL_DELTA), (float(e.max()), np.unravel_index(np.argmax(e), e.shape))
    C_ref = oracle.cls_tensor(k, D_ref, P_t, real="f80")
    e_auto, e_te = cl_err(C, C_ref)
    assert e_auto <= TOL_CL and e_te <= TOL_CL
    plan.close()


def test_tensor_at_the_papers_tensor_grid_sizes(los):
    """l = 2..1500 (l_max_tensor), k tau0 up to 3000 (k_eta_max_tensor), config-1 tau grid (1200 points)."""
    l_list = np.arange(2, 1501, dtype=np.int32)
    k = synth.k_grid(1000, 1e-5, 3000.0 / TAU0)
    tau = synth.tau_grid(600, 600, TAU0)
    S = tensor_sources(k, tau)
    P_t = 2.1e-10 * (k / 0.05) ** -0.01
    plan, D, C = run_tensor(los, l_list, k, tau, S, P_t)
    D_ref = oracle.transfer_tensor(l_list, k, tau, TAU0, *S, real="f80")
    C_ref = oracle.cls_tensor(k, D_ref, P_t, real="f80")
    e = delta_err(D, D_ref)
    print(f"tensor 1500 x 1000 x 1200: max Delta error per source {e.max(axis=1)}")
    assert np.all(e <= TOL_DELTA)
    e_auto, e_te = cl_err(C, C_ref)
    assert e_auto <= TOL_CL and e_te <= TOL_CL
    # spectra on every l from a CAMB-like sparse list of the same plan family (reading R25 on tensor spectra)
    l_sparse = np.unique(np.concatenate([np.arange(2, 40), np.arange(40, 200, 10), np.arange(200, 1501, 50), [1500]])).astype(np.int32)
    plan_s = los.Plan(l_sparse, k, tau, TAU0, tensor=True)
    d_S = [dev(s) for s in S]
    D_s = plan_s.gcamb_los_transfer_tensor(*d_S)
    rows = torch.from_numpy(l_sparse.astype(np.int64) - 2).cuda()
    # same sums, but the union list of a sparse plan puts the rows into other l-tiles: rounding-level agreement
    assert float((D_s - torch.from_numpy(D).cuda()[:, rows, :]).abs().max()) <= 1e-13 * float(np.abs(D).max())
    C_s = plan_s.gcamb_los_cls_tensor(D_s, dev(P_t))
    C_all = plan_s.gcamb_los_cl_interp(C_s).cpu().numpy()
    ref_all = oracle.cl_interp(l_sparse, oracle.cls_tensor(k, D_ref[:, l_sparse - 2, :], P_t, real="f80"), real="f80")
    assert C_all.shape == ref_all.shape == (4, 1499)
    l_all = np.arange(2, 1501, dtype=np.float64)
    dy = np.abs(C_all - ref_all) * l_all * (l_all + 1.0)
    assert np.all(np.max(dy, axis=-1) <= 1e-8 * np.max(np.abs(ref_all) * l_all * (l_all + 1.0), axis=-1))
    plan.close()
    plan_s.close()


def test_tensor_batched_equals_a_loop_of_single_calls(los):
    """a5 for the tensor calls: B cosmologies on one plan go out as ONE launch of the transfer kernels with 2 B
    members; Delta and C_l equal a loop of single calls bit for bit, and the oracle within the bars."""
    l_list = np.array([2, 3, 4, 9, 10, 30, 31, 32, 77, 150, 151, 260], dtype=np.int32)
    k = synth.k_grid(45, 1e-4, 0.04)
    tau = synth.tau_grid(150, 83, TAU0)
    B = 3
    S = [tensor_sources(k, tau, seed=77 + c) for c in range(B)]
    hS = [np.stack([S[c][q] for c in range(B)]) for q in range(3)]
    hP = np.stack([2.1e-10 * (1.0 + 0.1 * c) * (k / 0.05) ** (-0.01 * (c + 1)) for c in range(B)])
    plan = los.Plan(l_list, k, tau, TAU0, tensor=True)
    D = torch.full((B, 3, plan.n_l, plan.n_k), float("nan"), dtype=torch.float64, device="cuda")
    plan.gcamb_los_transfer_tensor_batched(dev(hS[0]), dev(hS[1]), dev(hS[2]), out=D)
    C = plan.gcamb_los_cls_tensor_batched(D, dev(hP))
    torch.cuda.synchronize()
    assert C.shape == (B, 4, plan.n_l)
    for c in range(B):
        D1 = plan.gcamb_los_transfer_tensor(dev(S[c][0]), dev(S[c][1]), dev(S[c][2]))
        C1 = plan.gcamb_los_cls_tensor(D1, dev(hP[c]))
        assert torch.equal(D1, D[c]) and torch.equal(C1, C[c])
    D_ref = oracle.transfer_tensor(l_list, k, tau, TAU0, *S[2], real="f80")
    assert np.all(delta_err(D[2].cpu().numpy(), D_ref) <= TOL_DELTA)
    e_auto, e_te = cl_err(C[2].cpu().numpy(), oracle.cls_tensor(k, D_ref, hP[2], real="f80"))
    assert e_auto <= TOL_CL and e_te <= TOL_CL
    # spectra of the batch on every l (reading R25)
    C_all = plan.gcamb_los_cl_interp(C)
    assert C_all.shape == (B, 4, 259)
    assert torch.equal(C_all[1], plan.gcamb_los_cl_interp(C[1].contiguous()))
    with pytest.raises(ValueError):                                # scratch of one cosmology for three
        plan.gcamb_los_transfer_tensor_batched(dev(hS[0]), dev(hS[1]), dev(hS[2]),
                                               work=torch.zeros(plan.gcamb_los_tensor_work_bytes() // 8, dtype=torch.float64, device="cuda"))
    plan.close()


def test_scalar_and_tensor_calls_do_not_mix(los):
    k = synth.k_grid(8, 1e-4, 0.01)
    tau = np.linspace(100.0, 13000.0, 40)
    l_list = np.arange(2, 20, dtype=np.int32)
    tplan = los.Plan(l_list, k, tau, TAU0, tensor=True)
    splan = los.Plan(l_list, k, tau, TAU0)
    z = torch.zeros(8, 40, dtype=torch.float64, device="cuda")
    with pytest.raises(los.GcambError) as e:
        tplan.gcamb_los_transfer(z, z, z)
    assert e.value.status == 1 and "tensor" in str(e.value)
    with pytest.raises(los.GcambError) as e:
        splan.gcamb_los_transfer_tensor(z, z, z, work=torch.zeros(16, dtype=torch.float64, device="cuda"))
    assert e.value.status == 1
    with pytest.raises(los.GcambError) as e:
        splan.gcamb_los_tensor_work_bytes()
    assert e.value.status == 1
    with pytest.raises(los.GcambError):
        los.Plan(np.array([65534], dtype=np.int32), k, tau, TAU0, tensor=True)      # l + 2 would not fit
    tplan.close()
    splan.close()


# --------------------------------------------------------------------------- InterpolateSources
@pytest.mark.parametrize("shape", [(40, 300, 181, (2,)), (2, 17, 40, ()), (3, 50, 1200, (3, 2)), (257, 3000, 600, (2,))])
def test_interp_sources_against_the_oracle(los, shape):
    n_kc, n_k, n_tau, lead = shape
    rng = np.random.default_rng(n_kc + n_k)
    kc = np.sort(np.concatenate([[1e-5, 0.6], rng.uniform(1e-5, 0.6, n_kc - 2)]))
    n_knots = min(3, n_kc - 2, n_k - 2)          # some fine k sit exactly on knots, and on both ends
    k = np.unique(np.concatenate([kc[[0, -1]], kc[1:-1][:n_knots], rng.uniform(kc[0], kc[-1], n_k - 2 - n_knots)]))
    assert k.size == n_k
    tau = np.linspace(100.0, 13900.0, n_tau)
    plan = los.Plan(np.arange(2, 10, dtype=np.int32), k, tau, TAU0)
    si = los.SourceInterp(plan, kc)
    S_c = np.cos(30.0 * kc[:, None] * (1.0 + np.arange(n_tau)[None, :] / n_tau)) * np.exp(-(kc[:, None] / 0.3) ** 2)
    S_c = S_c * (1.0 + 0.01 * rng.standard_normal(lead + S_c.shape))
    out = torch.full(lead + (n_k, n_tau), float("nan"), dtype=torch.float64, device="cuda")
    si.gcamb_los_interp_sources(dev(S_c), out=out)
    torch.cuda.synchronize()
    got = out.cpu().numpy().reshape((-1, n_k, n_tau))
    for s, Sc in enumerate(S_c.reshape((-1, n_kc, n_tau))):
        ref = oracle.interp_sources(kc, k, Sc, real="f80")
        assert np.max(np.abs(got[s] - ref)) <= 1e-13 * np.max(np.abs(Sc))
    assert torch.equal(out, si.gcamb_los_interp_sources(dev(S_c)))
    si.close()
    plan.close()


@pytest.mark.parametrize("case", [
    # (n_kc, n_k, n_tau, grid, banded): the solve runs with the banded inverse on the FP64 tensor cores, except for
    # grids of fewer than 3 or more than 4096 coarse wavenumbers, which keep the sequential sweeps
    (300, 900, 200, "log", True),
    (9, 30, 33, "log", True),                 # one block of 8 rows + 1, odd n_tau: scalar evaluation kernel
    (400, 300, 64, "alternating", True),      # spacings that jump by a factor 100 from one interval to the next
    (4097, 200, 40, "log", False),
    (2, 40, 32, "log", False),
])
def test_interp_sources_both_forms_of_the_solve(los, case):
    n_kc, n_k, n_tau, grid, banded = case
    if grid == "log":
        kc = synth.k_grid(n_kc, 1e-5, 0.6)
    else:
        kc = 1e-4 + np.concatenate([[0.0], np.cumsum(np.where(np.arange(n_kc - 1) % 2 == 0, 1e-5, 1e-3))])
    rng = np.random.default_rng(n_kc)
    k = np.sort(np.concatenate([kc[[0, -1]], rng.uniform(kc[0], kc[-1], n_k - 2)]))
    tau = np.linspace(100.0, 13900.0, n_tau)
    plan = los.Plan(np.arange(2, 10, dtype=np.int32), k, tau, TAU0)
    si = los.SourceInterp(plan, kc)
    assert (si.band_columns > 0) == banded and si.band_columns <= 100
    S_c = np.cos(30.0 * kc[:, None] * (1.0 + np.arange(n_tau)[None, :] / n_tau)) * np.exp(-(kc[:, None] / 0.3) ** 2)
    S_c = S_c * (1.0 + 0.01 * rng.standard_normal((2,) + S_c.shape))
    out = torch.full((2, n_k, n_tau), float("nan"), dtype=torch.float64, device="cuda")
    si.gcamb_los_interp_sources(dev(S_c), out=out)
    torch.cuda.synchronize()
    got = out.cpu().numpy()
    for s in range(2):
        ref = oracle.interp_sources(kc, k, S_c[s], real="f80")
        assert np.max(np.abs(got[s] - ref)) <= 1e-13 * np.max(np.abs(S_c[s]))
    assert torch.equal(out, si.gcamb_los_interp_sources(dev(S_c)))          # deterministic
    # an unaligned output buffer takes the scalar evaluation kernel: same values
    if n_tau % 2 == 0:
        buf = torch.empty(2 * n_k * n_tau + 1, dtype=torch.float64, device="cuda")
        out2 = buf[1:].view(2, n_k, n_tau)
        si.gcamb_los_interp_sources(dev(S_c), out=out2)
        assert torch.equal(out2, out)
    si.close()
    plan.close()


def test_interp_sources_captures_into_a_cuda_graph(los):
    """The call only enqueues its two kernels (the second one as a programmatic dependent launch of the first), so
    it can be captured once and replayed on new coarse sources, with caller scratch or with the static scratch."""
    kc = synth.k_grid(50, 1e-5, 0.6)
    k = synth.k_grid(333, 1e-5, 0.6)
    tau = np.linspace(100.0, 13900.0, 96)
    plan = los.Plan(np.arange(2, 10, dtype=np.int32), k, tau, TAU0)
    si = los.SourceInterp(plan, kc)
    rng = np.random.default_rng(3)
    d_S = dev(rng.standard_normal((2, 50, 96)))
    work = torch.empty_like(d_S)
    out = torch.empty(2, 333, 96, dtype=torch.float64, device="cuda")
    out_static = torch.empty_like(out)
    si.gcamb_los_interp_sources(d_S, out=out, work=work)
    si.gcamb_los_interp_sources_noalloc(d_S, out_static)           # first call on the device: outside the capture
    torch.cuda.synchronize()
    graph, side = torch.cuda.CUDAGraph(), torch.cuda.Stream()
    with torch.cuda.stream(side):
        with torch.cuda.graph(graph, stream=side):
            si.gcamb_los_interp_sources(d_S, out=out, work=work)
            si.gcamb_los_interp_sources_noalloc(d_S, out_static)
    for _ in range(2):
        d_S.copy_(dev(rng.standard_normal((2, 50, 96))))
        out.fill_(float("nan")); out_static.fill_(float("nan"))
        graph.replay()
        torch.cuda.synchronize()
        want = si.gcamb_los_interp_sources(d_S)
        assert torch.equal(out, want) and torch.equal(out_static, want)
    si.close()
    plan.close()


def test_interp_sources_feeds_the_transfer_kernel(los):
    """coarse sources -> InterpolateSources -> transfer -> C_l on the GPU against the same chain of the oracle."""
    cfg = synth.Config(9, "coarse-to-fine", 2, 300, 200, 1e-4, 0.05, 120, 60, False)
    k, tau = cfg.k(), cfg.tau()
    kc = synth.k_grid(60, 1e-4, 0.05)
    coarse = synth.Config(9, "coarse", 2, 300, 60, 1e-4, 0.05, 120, 60, False)
    S_Tc, S_Ec, _ = synth.sources(coarse, noise=False)          # smooth in k: what a spline can follow
    plan = los.Plan(cfg.l_list(), k, tau, cfg.tau0)
    si = los.SourceInterp(plan, kc)
    S_f = si.gcamb_los_interp_sources(dev(np.stack([S_Tc, S_Ec])))
    D = plan.gcamb_los_transfer(S_f[0], S_f[1])
    P = synth.primordial_power(cfg)
    C = plan.gcamb_los_cls(D, dev(P)).cpu().numpy()
    r_T, r_E = oracle.interp_sources(kc, k, S_Tc, real="f80"), oracle.interp_sources(kc, k, S_Ec, real="f80")
    D_ref = oracle.transfer(cfg.l_list(), k, tau, cfg.tau0, r_T, r_E, real="f80")
    C_ref = oracle.cls(k, D_ref, P, real="f80")
    e = delta_err(D.cpu().numpy(), D_ref)
    assert np.all(e <= TOL_DELTA)
    assert np.max(np.abs(C[:2] / C_ref[:2] - 1.0)) <= TOL_CL
    assert np.max(np.abs(C[2] - C_ref[2]) / np.sqrt(C_ref[2] ** 2 + C_ref[0] * C_ref[1])) <= TOL_CL
    # and the spline itself recovers the smooth sources of the fine grid to the accuracy the grid allows
    S_T_true, _, _ = synth.sources(cfg, noise=False)
    assert np.max(np.abs(S_f[0].cpu().numpy() - S_T_true)) <= 0.1 * np.max(np.abs(S_T_true))
    si.close()
    plan.close()


def test_interp_sources_error_paths(los):
    k = synth.k_grid(8, 1e-3, 0.01)
    tau = np.linspace(100.0, 13000.0, 10)
    plan = los.Plan(np.arange(2, 6, dtype=np.int32), k, tau, TAU0)
    with pytest.raises(los.GcambError) as e:
        los.SourceInterp(plan, np.array([2e-3, 0.02]))             # fine k below the coarse grid
    assert e.value.status == 2
    with pytest.raises(los.GcambError) as e:
        los.SourceInterp(plan, np.array([1e-3, 5e-3, 4e-3, 0.01]))   # not increasing
    assert e.value.status == 2
    with pytest.raises(los.GcambError) as e:
        los.SourceInterp(plan, np.array([1e-3]))
    assert e.value.status == 1
    plan.close()
