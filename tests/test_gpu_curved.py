"""SURVEY 8(f) NEXT-4 on the GPU: line-of-sight integration in OPEN and CLOSED universes (hyperspherical
Bessel functions, reading R28), element by element against the long-double oracle
(pinned in tests/test_oracle_curved.py).

Bars as for the flat path: |dDelta| <= 1e-10 max_k|Delta_l| per (source, l); C_l 1e-8 (R13).
Inputs: BASELINE.json's seeded synthetic source model on reduced grids; curvature radii from strongly
open (r_c = 6000 Mpc: chi up to 2.3, where Phi_l decays in l like tanh(chi/2)^l only) to nearly flat.
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


def delta_err(D_gpu, D_ref):
    scale = np.max(np.abs(D_ref), axis=-1)
    err = np.max(np.abs(D_gpu - D_ref), axis=-1)
    return err / np.where(scale > 0, scale, 1.0)


def cl_err(C_gpu, C_ref):
    auto = [0, 1] + ([3] if C_ref.shape[-2] == 4 else [])
    e_auto = float(np.max(np.abs(C_gpu[..., auto, :] / C_ref[..., auto, :] - 1.0)))
    norm = np.sqrt(C_ref[..., 2, :] ** 2 + C_ref[..., 0, :] * C_ref[..., 1, :])
    e_te = float(np.max(np.abs(C_gpu[..., 2, :] - C_ref[..., 2, :]) / norm))
    return e_auto, e_te


@pytest.mark.parametrize("case", [
    # (l_max, n_k, k_hi, n_tau_uniform, n_tau_log, with_phi, r_c)
    (200, 60, 0.02, 120, 60, False, 20000.0),
    (300, 48, 0.05, 200, 100, True, 9000.0),
    (150, 40, 0.01, 40, 29, False, 6000.0),        # chi up to 2.3: slow decay above the turning point
    (120, 33, 0.3, 90, 43, True, 30000.0),         # x far above l_max: every point starts at the top tile
    (260, 25, 0.03, 900, 700, False, 15000.0),     # 1600 tau: one pass of 256 threads
    (90, 9, 0.02, 1900, 1700, True, 12000.0),      # 3600 tau: several passes
    (200, 30, 0.02, 120, 60, False, 1.0e7),        # nearly flat
])
def test_open_universe_against_the_oracle(los, case):
    l_max, n_k, k_hi, n_u, n_log, with_phi, r_c = case
    cfg = synth.Config(9, "open", 2, l_max, n_k, 1e-4, k_hi, n_u, n_log, with_phi)
    K = -1.0 / r_c ** 2
    k, tau = cfg.k(), cfg.tau()
    S_T, S_E, S_P = synth.sources(cfg)
    P = synth.primordial_power(cfg)
    plan = los.Plan(cfg.l_list(), k, tau, cfg.tau0, with_phi=with_phi, curvature_K=K)
    D = torch.full((plan.n_src, plan.n_l, plan.n_k), float("nan"), dtype=torch.float64, device="cuda")
    C = torch.full((plan.n_spec, plan.n_l), float("nan"), dtype=torch.float64, device="cuda")
    d_S = (dev(S_T), dev(S_E), None if S_P is None else dev(S_P))
    plan.gcamb_los_transfer(*d_S, out=D)
    plan.gcamb_los_cls(D, dev(P), out=C)
    torch.cuda.synchronize()
    assert torch.equal(D, plan.gcamb_los_transfer(*d_S))                     # deterministic
    D, C = D.cpu().numpy(), C.cpu().numpy()
    assert np.all(np.isfinite(D)) and np.all(np.isfinite(C))
    D_ref = oracle.transfer_open(cfg.l_list(), k, tau, cfg.tau0, K, S_T, S_E, S_P, real="f80")
    C_ref = oracle.cls(k, D_ref, P, real="f80")
    e = delta_err(D, D_ref)
    assert np.all(e <= TOL_DELTA), (float(e.max()), np.unravel_index(np.argmax(e), e.shape))
    e_auto, e_te = cl_err(C, C_ref)
    assert e_auto <= TOL_CL and e_te <= TOL_CL
    if r_c >= 1.0e7:    # and the flat kernels are close by: the difference falls like |K|
        flat = los.Plan(cfg.l_list(), k, tau, cfg.tau0, with_phi=with_phi)
        D_flat = flat.gcamb_los_transfer(*d_S).cpu().numpy()
        assert np.max(np.abs(D_flat - D)) <= 1e-4 * np.max(np.abs(D))
        flat.close()
    plan.close()


def test_open_universe_batched_host_and_sparse_l(los):
    cfg = synth.Config(9, "open-batch", 2, 240, 70, 1e-4, 0.03, 120, 60, False, n_batch=3)
    K = -1.0 / 11000.0 ** 2
    plan = los.Plan(cfg.l_list(), cfg.k(), cfg.tau(), cfg.tau0, curvature_K=K)
    S = [synth.sources(cfg, c) for c in range(3)]
    hT, hE = np.stack([s[0] for s in S]), np.stack([s[1] for s in S])
    hP = np.stack([synth.primordial_power(cfg, c) for c in range(3)])
    Db = plan.gcamb_los_transfer_batched(dev(hT), dev(hE))
    Cb = plan.gcamb_los_cls_batched(Db, dev(hP))
    for c in range(3):
        D1 = plan.gcamb_los_transfer(dev(hT[c]), dev(hE[c]))
        assert torch.equal(D1, Db[c])
        D_ref = oracle.transfer_open(cfg.l_list(), cfg.k(), cfg.tau(), cfg.tau0, K, hT[c], hE[c], real="f80")
        assert np.all(delta_err(Db[c].cpu().numpy(), D_ref) <= TOL_DELTA)
    # the fused call takes the two-kernel path on a curved plan; the host entry point works as on a flat one
    info = plan.gcamb_los_spectra_batched_info(3)
    assert not info["fused"]
    Cs = plan.gcamb_los_spectra_batched(dev(hT), dev(hE), None, dev(hP))
    assert torch.equal(Cs, Cb)
    hC = np.empty((3, 3, cfg.n_l))
    plan.gcamb_los_spectra_host(hT, hE, None, hP, hC)
    assert np.array_equal(hC, Cb.cpu().numpy())
    # sparse l list: the dense kernels store the listed l only
    l_sparse = np.array([2, 3, 7, 20, 21, 100, 239, 240], dtype=np.int32)
    sp = los.Plan(l_sparse, cfg.k(), cfg.tau(), cfg.tau0, curvature_K=K)
    D_sp = sp.gcamb_los_transfer(dev(hT[0]), dev(hE[0]))
    rows = torch.from_numpy(l_sparse.astype(np.int64) - 2).cuda()
    assert torch.equal(D_sp, Db[0][:, rows, :])
    sp.close()
    plan.close()


def test_open_universe_at_config1_tau_grid(los):
    """l = 2..1000, 300 k, the 1200-point tau grid of config 1, Omega_K ~ 0.1 (r_c = 14000 Mpc)."""
    cfg = synth.Config(9, "open-1200", 2, 1000, 300, 1e-5, 0.12, 600, 600, False)
    K = -1.0 / 14000.0 ** 2
    S_T, S_E, _ = synth.sources(cfg)
    P = synth.primordial_power(cfg)
    plan = los.Plan(cfg.l_list(), cfg.k(), cfg.tau(), cfg.tau0, curvature_K=K)
    D = plan.gcamb_los_transfer(dev(S_T), dev(S_E))
    C = plan.gcamb_los_cls(D, dev(P)).cpu().numpy()
    D_ref = oracle.transfer_open(cfg.l_list(), cfg.k(), cfg.tau(), cfg.tau0, K, S_T, S_E, real="f80")
    C_ref = oracle.cls(cfg.k(), D_ref, P, real="f80")
    e = delta_err(D.cpu().numpy(), D_ref)
    print(f"open universe 999 x 300 x 1200: max Delta error per source {e.max(axis=1)}")
    assert np.all(e <= TOL_DELTA)
    e_auto, e_te = cl_err(C, C_ref)
    assert e_auto <= TOL_CL and e_te <= TOL_CL
    plan.close()


def closed_k_grid(n_k, beta_lo, beta_hi, r_c):
    """k = beta / r_c on n_k distinct integers beta, roughly log-spaced between beta_lo and beta_hi."""
    beta = np.unique(np.rint(np.geomspace(beta_lo, beta_hi, 3 * n_k)).astype(np.int64))
    beta = beta[np.linspace(0, beta.size - 1, n_k).astype(int)]
    return beta, beta / r_c


def closed_sources(cfg, k):
    """BASELINE.json's source model evaluated on the quantised k grid of a closed universe (seeded noise)."""
    tau = cfg.tau()[None, :]
    kk = k[:, None]
    g = np.exp(-((tau - 280.0) ** 2) / (2.0 * 20.0 ** 2)) / (20.0 * np.sqrt(2.0 * np.pi))
    damp = np.exp(-((kk / 0.1) ** 2))
    S_T = g * np.cos(kk * tau / np.sqrt(3.0)) * damp + 2.0 * np.exp(-(((tau - 11000.0) / 2000.0) ** 2)) * np.exp(-kk / 0.01)
    S_E = g * kk * np.sin(kk * tau / np.sqrt(3.0)) * damp
    S_P = np.exp(-(((tau - 9000.0) / 3000.0) ** 2)) * kk ** -2.0 * np.exp(-kk / 0.2) * np.ones_like(S_T)
    out = []
    for q, S in enumerate((S_T, S_E, S_P)):
        u = synth.uniform_pm1(cfg.seed, 700 + q, 0, S.size).reshape(S.shape)
        out.append(np.ascontiguousarray(S * (1.0 + 1e-3 * u)))
    return out


@pytest.mark.parametrize("case", [
    # (l_max, n_k, beta_lo, beta_hi, n_tau_uniform, n_tau_log, with_phi, r_c): r_c >= 2 tau0/pi keeps chi <= pi/2
    (200, 50, 3, 400, 120, 60, False, 12000.0),        # many rows end below l_max: Delta_l = 0 for l >= beta
    (300, 40, 3, 2500, 200, 100, True, 9000.0),        # chi up to 1.54
    (120, 30, 100, 6000, 90, 43, True, 30000.0),       # every row starts at the top tile
    (90, 12, 3, 60, 1900, 1700, False, 15000.0),       # several tau passes; beta - 1 below l_max on every row
    (200, 25, 50, 40000, 120, 60, False, 2.0e6),       # nearly flat
])
def test_closed_universe_against_the_oracle(los, case):
    l_max, n_k, b_lo, b_hi, n_u, n_log, with_phi, r_c = case
    cfg = synth.Config(9, "closed", 2, l_max, n_k, 1e-4, 0.1, n_u, n_log, with_phi)
    K = 1.0 / r_c ** 2
    beta, k = closed_k_grid(n_k, b_lo, b_hi, r_c)
    tau = cfg.tau()
    S_T, S_E, S_P = closed_sources(cfg, k)
    if not with_phi:
        S_P = None
    P = 2.1e-9 * (k / 0.05) ** -0.035
    plan = los.Plan(cfg.l_list(), k, tau, cfg.tau0, with_phi=with_phi, curvature_K=K)
    D = torch.full((plan.n_src, plan.n_l, plan.n_k), float("nan"), dtype=torch.float64, device="cuda")
    d_S = (dev(S_T), dev(S_E), None if S_P is None else dev(S_P))
    plan.gcamb_los_transfer(*d_S, out=D)
    C = plan.gcamb_los_cls(D, dev(P))
    torch.cuda.synchronize()
    assert torch.equal(D, plan.gcamb_los_transfer(*d_S))
    D, C = D.cpu().numpy(), C.cpu().numpy()
    assert np.all(np.isfinite(D)) and np.all(np.isfinite(C))
    D_ref = oracle.transfer_curved(cfg.l_list(), k, tau, cfg.tau0, K, S_T, S_E, S_P, real="f80")
    e = delta_err(D, D_ref)
    assert np.all(e <= TOL_DELTA), (float(e.max()), np.unravel_index(np.argmax(e), e.shape))
    # Phi_l^beta = 0 for l >= beta: exact zeros, on both sides
    above = cfg.l_list()[None, :, None] >= beta[None, None, :]
    assert np.all(D[np.broadcast_to(above, D.shape)] == 0.0) and np.all(D_ref[np.broadcast_to(above, D.shape)] == 0.0)
    C_ref = oracle.cls(k, D_ref, P, real="f80")
    live = cfg.l_list() < beta.max()              # above the largest beta every transfer function, hence C_l, is 0
    assert np.all(C[:, ~live] == 0.0) and np.all(C_ref[:, ~live] == 0.0)
    e_auto, e_te = cl_err(C[:, live], C_ref[:, live])
    assert e_auto <= TOL_CL and e_te <= TOL_CL
    plan.close()


@pytest.mark.parametrize("seed", range(16))
def test_random_small_curved_shapes(los, seed):
    """Seeded random grids, l lists, curvature radii and batch sizes around the kernel's shape boundaries, open
    (even seeds) and closed (odd seeds) universes, element by element against the long-double oracle; the bar
    carries the skip rule's own allowance (1e-30 sum |w S|) where Delta_l lies below the cut (cf. the flat test)."""
    rng = np.random.default_rng(5000 + seed)
    closed = bool(seed % 2)
    tau0 = 14000.0
    n_tau = int(rng.choice([2, 3, 32, 33, 127, 129, 300, 641, 1537, 2600]))
    tau = np.unique(np.sort(rng.uniform(10.0, 13990.0, n_tau)))
    r_c = float(rng.choice([9500.0, 12000.0, 20000.0, 60000.0])) if closed else float(rng.choice([5000.0, 9000.0, 20000.0, 3.0e5]))
    n_k = int(rng.integers(2, 12))
    if closed:
        beta = np.unique(rng.integers(3, int(rng.choice([40, 400, 4000])), n_k))
        k = beta / r_c
        K = 1.0 / r_c ** 2
    else:
        k = np.unique(np.sort(float(rng.choice([1e-3, 0.02, 0.2])) * rng.uniform(1e-3, 1.0, n_k)))
        K = -1.0 / r_c ** 2
    n_k = k.size
    if n_k < 2:
        pytest.skip("degenerate draw")
    with_phi = bool(rng.integers(0, 2))
    B = int(rng.choice([1, 1, 2, 3]))
    l_lo = int(rng.choice([2, 2, 17, 300]))
    l_all = np.arange(l_lo, l_lo + int(rng.choice([0, 1, 7, 8, 9, 63, 200])) + 1)
    if rng.integers(0, 2) and l_all.size > 3:
        l_all = np.sort(rng.choice(l_all, size=max(2, l_all.size // int(rng.integers(2, 9))), replace=False))
    l_list = l_all.astype(np.int32)
    S = rng.standard_normal((3, B, n_k, tau.size)) * np.exp(rng.uniform(-20, 5, (3, B, n_k, 1)))
    plan = los.Plan(l_list, k, tau, tau0, with_phi=with_phi, curvature_K=K)
    n_src = 3 if with_phi else 2
    D = torch.full((B, n_src, l_list.size, n_k), float("nan"), dtype=torch.float64, device="cuda")
    plan.gcamb_los_transfer_batched(dev(S[0]), dev(S[1]), dev(S[2]) if with_phi else None, out=D)
    torch.cuda.synchronize()
    D = D.cpu().numpy()
    w = oracle.trapz_weights(tau)
    chi = (tau0 - tau) / r_c
    bs = (k * r_c)[:, None] * (np.sin(chi) if closed else np.sinh(chi))[None, :]
    pref = np.sqrt((l_list + 2.0) * (l_list + 1.0) * l_list * (l_list - 1.0))
    for c in range(B):
        D_ref = oracle.transfer_curved(l_list, k, tau, tau0, K, S[0, c], S[1, c], S[2, c] if with_phi else None, real="f80")
        skip = [np.sum(np.abs(w * S[0, c]), axis=1)[None, :] * np.ones((l_list.size, 1)),
                np.sum(np.abs(w * S[1, c]) / bs ** 2, axis=1)[None, :] * pref[:, None]]
        if with_phi:
            skip.append(np.sum(np.abs(w * S[2, c]), axis=1)[None, :] * np.ones((l_list.size, 1)))
        bound = TOL_DELTA * np.max(np.abs(D_ref), axis=-1, keepdims=True) + 1e-30 * np.stack(skip)
        assert np.all(np.isfinite(D[c]))
        assert np.all(np.abs(D[c] - D_ref) <= bound), (seed, closed, tau.size, n_k, with_phi, B, r_c, l_list[0], l_list[-1])
    plan.close()


def test_curved_plans_that_are_rejected(los):
    tau = np.linspace(100.0, 13000.0, 10)
    l_list = np.arange(2, 6, dtype=np.int32)
    r_c = 10000.0
    k_int = np.array([3.0, 4.0, 7.0, 12.0]) / r_c
    los.Plan(l_list, k_int, tau, 14000.0, curvature_K=1.0 / r_c ** 2).close()          # a valid closed plan
    with pytest.raises(los.GcambError) as e:
        los.Plan(l_list, np.array([3.0, 4.5, 7.0]) / r_c, tau, 14000.0, curvature_K=1.0 / r_c ** 2)
    assert e.value.status == 2 and "integer" in str(e.value)
    with pytest.raises(los.GcambError) as e:
        los.Plan(l_list, np.array([2.0, 4.0]) / r_c, tau, 14000.0, curvature_K=1.0 / r_c ** 2)        # beta < 3
    assert e.value.status == 2
    with pytest.raises(los.GcambError) as e:
        los.Plan(l_list, k_int * (r_c / 5000.0), tau, 14000.0, curvature_K=1.0 / 5000.0 ** 2)        # chi up to 2.8 > pi/2
    assert e.value.status == 2 and "pi/2" in str(e.value)
    with pytest.raises(los.GcambError) as e:
        los.Plan(l_list, k_int, tau, 14000.0, tensor=True, curvature_K=-1e-8)
    assert e.value.status == 1
