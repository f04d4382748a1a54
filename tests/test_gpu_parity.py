"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle on the same seeded inputs.

Bars (BASELINE.json north_star):  |Delta_GPU - Delta_oracle| <= 1e-10 * max_k |Delta_l|  per l and
source;  C_l relative error <= 1e-8 for TT, EE, phiphi; for TE, which crosses zero, the same bound
relative to sqrt(C_TE^2 + C_TT C_EE) (reading R13, the paper's own TE normaliser, Eq. 5
PAPER.md:237).  The grading oracle is the long-double build (R14); the fp64 build is checked too.
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


def delta_err(D_gpu, D_ref, scale=None):
    """max over (source, l) of max_k |diff| / max_k |Delta_l|."""
    if scale is None:
        scale = np.max(np.abs(D_ref), axis=-1, keepdims=True)
    scale = np.where(scale > 0, scale, 1.0)
    return float(np.max(np.abs(D_gpu - D_ref) / scale))


def cl_err(C_gpu, C_ref):
    auto = [0, 1] + ([3] if C_ref.shape[-2] == 4 else [])
    e_auto = float(np.max(np.abs(C_gpu[..., auto, :] / C_ref[..., auto, :] - 1.0)))
    norm = np.sqrt(C_ref[..., 2, :] ** 2 + C_ref[..., 0, :] * C_ref[..., 1, :])
    e_te = float(np.max(np.abs(C_gpu[..., 2, :] - C_ref[..., 2, :]) / norm))
    return e_auto, e_te


def run_gpu(los, l_list, k, tau, tau0, S_T, S_E, S_P, P_R):
    plan = los.Plan(l_list, k, tau, tau0, with_phi=S_P is not None)
    # NaN pre-fill: an element the kernels fail to write cannot pass
    D = torch.full((plan.n_src, plan.n_l, plan.n_k), float("nan"), dtype=torch.float64, device="cuda")
    C = torch.full((plan.n_spec, plan.n_l), float("nan"), dtype=torch.float64, device="cuda")
    plan.gcamb_los_transfer(dev(S_T), dev(S_E), None if S_P is None else dev(S_P), out=D)
    plan.gcamb_los_cls(D, dev(P_R), out=C)
    torch.cuda.synchronize()
    out = D.cpu().numpy(), C.cpu().numpy(), plan
    return out


# --------------------------------------------------------------------------- config 0, element by element
@pytest.mark.parametrize("real", ["f80", "f64"])
def test_config0_full_parity(los, real):
    cfg = synth.CONFIGS[0]
    S_T, S_E, _ = synth.sources(cfg)
    P = synth.primordial_power(cfg)
    D, C, plan = run_gpu(los, cfg.l_list(), cfg.k(), cfg.tau(), cfg.tau0, S_T, S_E, None, P)
    assert plan.nominal_terms == cfg.nominal_terms()
    assert 0 < plan.executed_terms < plan.nominal_terms
    D_ref = oracle.transfer(cfg.l_list(), cfg.k(), cfg.tau(), cfg.tau0, S_T, S_E, real=real)
    C_ref = oracle.cls(cfg.k(), D_ref, P, real=real)
    assert delta_err(D, D_ref) <= TOL_DELTA
    e_auto, e_te = cl_err(C, C_ref)
    assert e_auto <= TOL_CL and e_te <= TOL_CL
    # the C_l kernel alone, fed the oracle's Delta
    C2 = plan.gcamb_los_cls(dev(D_ref), dev(P)).cpu().numpy()
    e_auto, e_te = cl_err(C2, C_ref)
    assert e_auto <= 1e-13 and e_te <= 1e-13


# --------------------------------------------------------------------------- ragged / edge shapes
def _small_problem(n_l_spec, n_k, n_tau, with_phi, seed):
    rng = np.random.default_rng(seed)
    tau0 = 14000.0
    tau = np.sort(rng.uniform(50.0, 13990.0, n_tau))
    tau[-1] = 13999.5
    k = np.geomspace(3e-5, 0.11, n_k) * (1 + 0.01 * rng.uniform(-1, 1, n_k))
    k.sort()
    S = [rng.standard_normal((n_k, n_tau)) for _ in range(3)]
    P = rng.uniform(1e-9, 3e-9, n_k)
    return n_l_spec, k, tau, tau0, S[0], S[1], S[2] if with_phi else None, P


@pytest.mark.parametrize("case", [
    (np.arange(2, 200), 33, 97, False, 1),            # ragged tau (not a multiple of 32 or of the CTA)
    (np.arange(2, 77), 5, 2, True, 2),                # minimum n_tau
    (np.array([2]), 2, 40, False, 3),                 # single l, minimum n_k
    (np.array([5, 6, 40, 41, 300, 1500]), 17, 300, True, 4),    # sparse l list (R21), x up to 1540
    (np.arange(700, 900), 9, 130, False, 5),          # l range not starting at 2
    (np.arange(2, 40), 12, 1300, True, 6),            # n_tau just above 128 x 10
    (np.arange(2, 60), 6, 3100, False, 7),            # n_tau above one CTA's slots: three passes, n_src=2
    (np.arange(2, 230), 8, 300, False, 8),            # few rows: the launch trades points per thread for threads
])
def test_edge_shapes(los, case):
    l_list, k, tau, tau0, S_T, S_E, S_P, P = _small_problem(*case)
    l_list = np.asarray(l_list, dtype=np.int32)
    D, C, _ = run_gpu(los, l_list, k, tau, tau0, S_T, S_E, S_P, P)
    D_ref = oracle.transfer(l_list, k, tau, tau0, S_T, S_E, S_P, real="f80")
    C_ref = oracle.cls(k, D_ref, P, real="f80")
    assert D.shape == D_ref.shape and C.shape == C_ref.shape
    assert delta_err(D, D_ref) <= TOL_DELTA
    e_auto, e_te = cl_err(C, C_ref)
    assert e_auto <= TOL_CL and e_te <= TOL_CL


def test_batched_tau_passes_with_phi(los):
    """n_tau above one CTA's slots: the CTA takes the tau range in passes and adds each pass to what
    it stored before; batched, three sources, sparse l list; still equal to the single calls bit for bit."""
    rng = np.random.default_rng(11)
    n_k, n_tau, B = 7, 3300, 3
    tau = np.sort(rng.uniform(100.0, 13900.0, n_tau))
    k = np.geomspace(1e-4, 0.05, n_k)
    l_list = np.array([2, 3, 9, 10, 11, 64, 65, 200, 399, 640], dtype=np.int32)
    S = rng.standard_normal((3, B, n_k, n_tau))
    P = rng.uniform(1e-9, 3e-9, (B, n_k))
    plan = los.Plan(l_list, k, tau, 14000.0, with_phi=True)
    Db = torch.full((B, 3, l_list.size, n_k), float("nan"), dtype=torch.float64, device="cuda")
    plan.gcamb_los_transfer_batched(dev(S[0]), dev(S[1]), dev(S[2]), out=Db)
    Cb = plan.gcamb_los_cls_batched(Db, dev(P))
    for c in range(B):
        D1 = plan.gcamb_los_transfer(dev(S[0, c]), dev(S[1, c]), dev(S[2, c]))
        assert torch.equal(D1, Db[c])
        D_ref = oracle.transfer(l_list, k, tau, 14000.0, S[0, c], S[1, c], S[2, c], real="f80")
        C_ref = oracle.cls(k, D_ref, P[c], real="f80")
        assert delta_err(Db[c].cpu().numpy(), D_ref) <= TOL_DELTA
        e_auto, e_te = cl_err(Cb[c].cpu().numpy(), C_ref)
        assert e_auto <= TOL_CL and e_te <= TOL_CL
    plan.close()


@pytest.mark.parametrize("n_src", [2, 3])
def test_many_tau_passes_are_deterministic(los, n_src):
    """n_tau ~ 7000: five passes of one CTA per k (no atomics, no cleared output buffer).  Oracle
    parity, run-to-run bit equality on a NaN-prefilled buffer, batched == single."""
    rng = np.random.default_rng(21 + n_src)
    n_k, n_tau, B = 9, 7001, 2
    tau = np.sort(rng.uniform(100.0, 13950.0, n_tau))
    k = np.geomspace(2e-4, 0.06, n_k)
    l_list = np.arange(2, 420, dtype=np.int32)
    S = rng.standard_normal((3, B, n_k, n_tau))
    P = rng.uniform(1e-9, 3e-9, (B, n_k))
    plan = los.Plan(l_list, k, tau, 14000.0, with_phi=n_src == 3)
    args = lambda c=None: [dev(S[q] if c is None else S[q, c]) for q in range(n_src)] + [None] * (3 - n_src)
    runs = []
    for _ in range(3):
        Db = torch.full((B, n_src, l_list.size, n_k), float("nan"), dtype=torch.float64, device="cuda")
        plan.gcamb_los_transfer_batched(*args(), out=Db)
        runs.append(Db)
    assert torch.equal(runs[0], runs[1]) and torch.equal(runs[0], runs[2])
    for c in range(B):
        D1 = torch.full((n_src, l_list.size, n_k), float("nan"), dtype=torch.float64, device="cuda")
        plan.gcamb_los_transfer(*args(c), out=D1)
        assert torch.equal(D1, runs[0][c])
        D_ref = oracle.transfer(l_list, k, tau, 14000.0, S[0, c], S[1, c], S[2, c] if n_src == 3 else None, real="f80")
        assert delta_err(runs[0][c].cpu().numpy(), D_ref) <= TOL_DELTA
    plan.close()


@pytest.mark.parametrize("n_plain", [1, 2, 4])
def test_few_plain_rows_after_the_compensated_launch(los, n_plain):
    """All but 1..4 k rows lie above the compensation threshold (x_max = k chi_0 > 6755): the plain
    launch that overlaps the compensated one is tiny and would retire long before it.  Work that
    follows in the stream (here the C_l kernel and a device-side copy) must still see every row."""
    tau = np.concatenate([np.linspace(200.0, 400.0, 90), np.geomspace(420.0, 13999.0, 70)])
    k = np.concatenate([np.geomspace(1e-3, 0.2, n_plain), np.linspace(0.5, 0.9, 40)])
    assert np.sum(k * (14000.0 - tau[0]) > 6755.4) == 40
    l_list = np.arange(2, 900, dtype=np.int32)
    rng = np.random.default_rng(70 + n_plain)
    S_T, S_E = rng.standard_normal((2, k.size, tau.size))
    P = rng.uniform(1e-9, 3e-9, k.size)
    plan = los.Plan(l_list, k, tau, 14000.0)
    assert plan.transfer_launches == 2
    D_ref = oracle.transfer(l_list, k, tau, 14000.0, S_T, S_E, real="f80")
    C_ref = oracle.cls(k, D_ref, P, real="f80")
    d_T, d_E, d_P = dev(S_T), dev(S_E), dev(P)
    for _ in range(5):
        D = torch.full((2, l_list.size, k.size), float("nan"), dtype=torch.float64, device="cuda")
        C = torch.full((3, l_list.size), float("nan"), dtype=torch.float64, device="cuda")
        plan.gcamb_los_transfer(d_T, d_E, out=D)
        plan.gcamb_los_cls(D, d_P, out=C)
        D_copy = D.clone()
        torch.cuda.synchronize()
        assert delta_err(D_copy.cpu().numpy(), D_ref) <= TOL_DELTA
        e_auto, e_te = cl_err(C.cpu().numpy(), C_ref)
        assert e_auto <= TOL_CL and e_te <= TOL_CL
    plan.close()


def test_rows_that_never_start_and_rows_above_the_compensation_threshold(los):
    """l range far above x for the small k (their Delta rows are all zero, the CTA walks nothing)
    together with k rows whose x_max exceeds 6755 (compensated coefficient launch)."""
    tau = np.concatenate([np.linspace(200.0, 400.0, 70), np.geomspace(420.0, 13999.0, 50)])
    k = np.concatenate([np.geomspace(1e-5, 1e-3, 6), np.linspace(0.3, 0.62, 9)])
    l_list = np.arange(1500, 1640, dtype=np.int32)
    rng = np.random.default_rng(5)
    S_T, S_E = rng.standard_normal((2, k.size, tau.size))
    P = np.full(k.size, 2e-9)
    D, C, plan = run_gpu(los, l_list, k, tau, 14000.0, S_T, S_E, None, P)
    assert plan.transfer_launches == 2
    assert np.all(D[:, :, :6] == 0.0)                      # x <= 14 there, l >= 1500
    D_ref = oracle.transfer(l_list, k, tau, 14000.0, S_T, S_E, real="f80")
    assert delta_err(D, D_ref) <= TOL_DELTA
    plan.close()


def test_single_tau_source_is_the_kernel(los):
    """P3 on the GPU: S = delta_{i,i*}/w_{i*} gives Delta_l(k) = j_l(k chi*) (values: oracle column)."""
    tau = np.array([100.0, 280.0, 700.0, 13000.0])
    k = np.geomspace(2e-4, 0.2, 50)
    S = np.zeros((k.size, tau.size)); S[:, 1] = 1.0 / 300.0
    l_list = np.arange(2, 1200, dtype=np.int32)
    D, _, _ = run_gpu(los, l_list, k, tau, 14000.0, S, S, S, np.ones(k.size))
    for j in (0, 13, 37, 49):
        x = float(k[j] * (14000.0 - 280.0))
        jl = oracle.sph_bessel(x, 1199, real="f80")[2:]
        assert np.max(np.abs(D[0, :, j] - jl)) <= 3e-12 / max(x, 1.0) + 1e-300
        assert np.array_equal(D[2, :, j], D[0, :, j])

# --------------------------------------------------------------------------- C_l kernels alone (a4)
@pytest.mark.parametrize("shape", [
    # (n_k, n_l, batch, with_phi): the streaming kernel (n_k even, <= 6144) at its chunk boundaries,
    # with more rows than SMs, fewer rows than SMs, CTA row ranges that straddle cosmologies;
    # the row-per-CTA kernel for odd and long rows
    (1536, 40, 1, False), (1538, 7, 3, True), (3000, 300, 1, False), (3072, 33, 5, False),
    (6144, 12, 2, True), (2, 9, 4, False), (50, 700, 3, True),
    (6146, 10, 2, False), (1537, 21, 2, True), (20000, 6, 1, True),
])
def test_cls_kernels_on_random_transfer_functions(los, shape):
    """Eq. 1 alone, on random Delta (no structure a wrong index could hide behind): element by element
    against the long-double oracle, batched == loop of single calls bit for bit, run-to-run bit equality."""
    n_k, n_l, B, with_phi = shape
    rng = np.random.default_rng(n_k + n_l)
    k = np.geomspace(1e-4, 0.5, n_k) * (1.0 + 0.1 * rng.uniform(size=n_k) / n_k)     # non-uniform ln k steps
    k = np.sort(k)
    tau = np.array([100.0, 5000.0, 13000.0])
    l_list = np.arange(2, 2 + n_l, dtype=np.int32)
    plan = los.Plan(l_list, k, tau, 14000.0, with_phi=with_phi)
    D = rng.standard_normal((B, plan.n_src, n_l, n_k))
    P = rng.uniform(1e-9, 3e-9, size=(B, n_k))
    d_D, d_P = dev(D), dev(P)
    C = torch.full((B, plan.n_spec, n_l), float("nan"), dtype=torch.float64, device="cuda")
    plan.gcamb_los_cls_batched(d_D, d_P, out=C)
    torch.cuda.synchronize()
    C_h = C.cpu().numpy()
    for b in range(B):
        C_ref = oracle.cls(k, D[b], P[b], real="f80")
        auto = [0, 1] + ([3] if with_phi else [])
        assert np.max(np.abs(C_h[b][auto] / C_ref[auto] - 1.0)) <= 1e-13
        norm = np.sqrt(C_ref[0] * C_ref[1])
        assert np.max(np.abs(C_h[b][2] - C_ref[2]) / norm) <= 1e-13
        assert torch.equal(plan.gcamb_los_cls(d_D[b], d_P[b]), C[b])
    assert torch.equal(plan.gcamb_los_cls_batched(d_D, d_P), C)
    plan.close()


# --------------------------------------------------------------------------- batched == loop of single
def test_batched_equals_loop_of_single(los):
    cfg = synth.Config(9, "mini-batch", 2, 300, 64, 1e-4, 0.25, 120, 60, False, n_batch=5)
    plan = los.Plan(cfg.l_list(), cfg.k(), cfg.tau(), cfg.tau0)
    S = [synth.sources(cfg, c) for c in range(cfg.n_batch)]
    S_T = dev(np.stack([s[0] for s in S])); S_E = dev(np.stack([s[1] for s in S]))
    P = dev(np.stack([synth.primordial_power(cfg, c) for c in range(cfg.n_batch)]))
    Db = plan.gcamb_los_transfer_batched(S_T, S_E)
    Cb = plan.gcamb_los_cls_batched(Db, P)
    for c in range(cfg.n_batch):
        D1 = plan.gcamb_los_transfer(S_T[c].contiguous(), S_E[c].contiguous())
        C1 = plan.gcamb_los_cls(D1, P[c].contiguous())
        assert torch.equal(D1, Db[c]) and torch.equal(C1, Cb[c])     # bit-exact: same kernels, same order
    D_ref = oracle.transfer(cfg.l_list(), cfg.k(), cfg.tau(), cfg.tau0, S[3][0], S[3][1], real="f80")
    assert delta_err(Db[3].cpu().numpy(), D_ref) <= TOL_DELTA


def test_host_buffer_entry_point_matches_device_path(los):
    cfg = synth.Config(9, "mini", 2, 150, 48, 1e-4, 0.2, 100, 50, True)
    plan = los.Plan(cfg.l_list(), cfg.k(), cfg.tau(), cfg.tau0, with_phi=True)
    S_T, S_E, S_P = synth.sources(cfg)
    P = synth.primordial_power(cfg)
    D = plan.gcamb_los_transfer(dev(S_T), dev(S_E), dev(S_P))
    C = plan.gcamb_los_cls(D, dev(P))
    Cl = np.empty((1, 4, cfg.n_l)); Dl = np.empty((1, 3, cfg.n_l, cfg.n_k))
    plan.gcamb_los_spectra_host(S_T[None], S_E[None], S_P[None], P[None], Cl, Dl)
    assert np.array_equal(Cl[0], C.cpu().numpy()) and np.array_equal(Dl[0], D.cpu().numpy())


@pytest.mark.parametrize("with_phi", [False, True])
def test_pipelined_host_entry_point_batched(los, with_phi):
    """n_k >= 64 and at least 4 MiB of sources: the sources go up in four blocks of k rows that overlap the
    kernels of the blocks before them; results must equal the device-resident path bit for bit, for a batch too."""
    cfg = synth.Config(9, "mini-pipe", 2, 400, 300, 1e-4, 0.25, 250, 150, with_phi, n_batch=3)
    assert 8 * cfg.n_k * cfg.n_tau * cfg.n_batch * (3 if with_phi else 2) >= 4 << 20
    plan = los.Plan(cfg.l_list(), cfg.k(), cfg.tau(), cfg.tau0, with_phi=with_phi)
    S = [synth.sources(cfg, c) for c in range(cfg.n_batch)]
    hS = [np.stack([s[q] for s in S]) if S[0][q] is not None else None for q in range(3)]
    hP = np.stack([synth.primordial_power(cfg, c) for c in range(cfg.n_batch)])
    D = plan.gcamb_los_transfer_batched(dev(hS[0]), dev(hS[1]), None if hS[2] is None else dev(hS[2]))
    C = plan.gcamb_los_cls_batched(D, dev(hP))
    Cl = np.full((cfg.n_batch, plan.n_spec, cfg.n_l), np.nan)
    Dl = np.full((cfg.n_batch, plan.n_src, cfg.n_l, cfg.n_k), np.nan)
    for _ in range(2):          # the second call reuses the plan's streams and scratch
        plan.gcamb_los_spectra_host(hS[0], hS[1], hS[2], hP, Cl, Dl)
        assert np.array_equal(Cl, C.cpu().numpy()) and np.array_equal(Dl, D.cpu().numpy())
    D_ref = oracle.transfer(cfg.l_list(), cfg.k(), cfg.tau(), cfg.tau0, S[1][0], S[1][1], S[1][2], real="f80")
    assert delta_err(Dl[1], D_ref) <= TOL_DELTA
    plan.close()


def test_transfer_and_cls_capture_into_a_cuda_graph(los):
    """The calls only enqueue work on the given stream (no allocation, no synchronisation), so a
    step can be captured once and replayed (emulator loops)."""
    cfg = synth.CONFIGS[0]
    S_T, S_E, _ = synth.sources(cfg)
    plan = los.Plan(cfg.l_list(), cfg.k(), cfg.tau(), cfg.tau0)
    d_T, d_E, d_P = dev(S_T), dev(S_E), dev(synth.primordial_power(cfg))
    D = torch.empty(2, cfg.n_l, cfg.n_k, dtype=torch.float64, device="cuda")
    C = torch.empty(3, cfg.n_l, dtype=torch.float64, device="cuda")
    plan.gcamb_los_transfer(d_T, d_E, out=D)
    plan.gcamb_los_cls(D, d_P, out=C)
    torch.cuda.synchronize()
    D0, C0 = D.clone(), C.clone()
    graph, side = torch.cuda.CUDAGraph(), torch.cuda.Stream()
    with torch.cuda.stream(side):
        with torch.cuda.graph(graph, stream=side):
            plan.gcamb_los_transfer(d_T, d_E, out=D)
            plan.gcamb_los_cls(D, d_P, out=C)
    for _ in range(2):
        D.fill_(float("nan"))
        C.fill_(float("nan"))
        graph.replay()
        torch.cuda.synchronize()
        assert torch.equal(D, D0) and torch.equal(C, C0)
    plan.close()


def test_errors_cross_the_abi_as_status_codes(los):
    cfg = synth.CONFIGS[0]
    with pytest.raises(los.GcambError) as e:
        los.Plan(cfg.l_list(), cfg.k()[::-1].copy(), cfg.tau(), cfg.tau0)
    assert e.value.status == 2
    with pytest.raises(los.GcambError) as e:
        los.Plan(cfg.l_list(), cfg.k(), cfg.tau(), cfg.tau()[-1])       # x = 0 (R18)
    assert e.value.status == 2
    with pytest.raises(los.GcambError) as e:
        los.Plan([1, 2, 3], cfg.k(), cfg.tau(), cfg.tau0)
    assert e.value.status == 1
    plan = los.Plan(cfg.l_list(), cfg.k(), cfg.tau(), cfg.tau0)
    z = torch.zeros(cfg.n_k, cfg.n_tau, dtype=torch.float64, device="cuda")
    with pytest.raises(los.GcambError) as e:
        plan.gcamb_los_transfer(z, z, z)                                # phi source without the mask bit
    assert e.value.status == 1


# --------------------------------------------------------------------------- seeded random shapes
@pytest.mark.parametrize("seed", range(32))
def test_random_small_shapes(los, seed):
    """Seeded random grids and l lists around the kernel's shape boundaries (one warp to several
    CTAs per k, dense and sparse l lists, l ranges far above or below x, with and without phi,
    with and without a batch), element by element against the long-double oracle.

    Unlike BASELINE.json's configs (k_max tau0 ~ 2 l_max) these l ranges may lie entirely above
    x + 18 x^(1/3) for every k, where Delta_l consists of nothing but terms the skip rule drops
    (R16: |j_l(x)| < 1e-30 may be skipped); the bar therefore carries the rule's own allowance,
    1e-30 sum_i |w_i S_X(k,tau_i)| (times the Delta^E factor), next to 1e-10 max_k |Delta_l|."""
    rng = np.random.default_rng(1000 + seed)
    n_tau = int(rng.choice([2, 3, 31, 32, 33, 64, 127, 128, 129, 300, 641, 1281, 1537, 2600]))
    n_k = int(rng.integers(2, 12))
    with_phi = bool(rng.integers(0, 2))
    B = int(rng.choice([1, 1, 2, 3]))
    tau0 = 14000.0
    tau = np.sort(rng.uniform(10.0, 13999.0, n_tau))
    tau = np.unique(tau)
    n_tau = tau.size
    k_hi = float(rng.choice([1e-3, 0.02, 0.2, 0.61]))
    k = np.sort(k_hi * rng.uniform(1e-3, 1.0, n_k))
    k = np.unique(k)
    n_k = k.size
    l_lo = int(rng.choice([2, 2, 17, 300, 1200]))
    l_hi = l_lo + int(rng.choice([0, 1, 7, 8, 9, 63, 200, 700]))
    l_all = np.arange(l_lo, l_hi + 1)
    if rng.integers(0, 2) and l_all.size > 3:
        l_all = np.sort(rng.choice(l_all, size=max(2, l_all.size // int(rng.integers(2, 9))), replace=False))
    l_list = l_all.astype(np.int32)
    S = rng.standard_normal((3, B, n_k, n_tau)) * np.exp(rng.uniform(-20, 5, (3, B, n_k, 1)))
    P = rng.uniform(1e-9, 3e-9, (B, n_k))
    plan = los.Plan(l_list, k, tau, tau0, with_phi=with_phi)
    n_src = 3 if with_phi else 2
    D = torch.full((B, n_src, l_list.size, n_k), float("nan"), dtype=torch.float64, device="cuda")
    C = torch.full((B, n_src + 1, l_list.size), float("nan"), dtype=torch.float64, device="cuda")
    plan.gcamb_los_transfer_batched(dev(S[0]), dev(S[1]), dev(S[2]) if with_phi else None, out=D)
    plan.gcamb_los_cls_batched(D, dev(P), out=C)
    torch.cuda.synchronize()
    D, C = D.cpu().numpy(), C.cpu().numpy()
    for c in range(B):
        D_ref = oracle.transfer(l_list, k, tau, tau0, S[0, c], S[1, c], S[2, c] if with_phi else None, real="f80")
        C_ref = oracle.cls(k, D_ref, P[c], real="f80")
        w = oracle.trapz_weights(tau)
        x = k[:, None] * (tau0 - tau)[None, :]
        pref = np.sqrt((l_list + 2.0) * (l_list + 1.0) * l_list * (l_list - 1.0))
        skip = [np.sum(np.abs(w * S[0, c]), axis=1)[None, :] * np.ones((l_list.size, 1)),
                np.sum(np.abs(w * S[1, c]) / x ** 2, axis=1)[None, :] * pref[:, None]]
        if with_phi:
            skip.append(np.sum(np.abs(w * S[2, c]), axis=1)[None, :] * np.ones((l_list.size, 1)))
        bound = TOL_DELTA * np.max(np.abs(D_ref), axis=-1, keepdims=True) + 1e-30 * np.stack(skip)
        assert np.all(np.abs(D[c] - D_ref) <= bound), (seed, n_tau, n_k, with_phi, B, l_lo, l_hi)
        big = np.max(np.abs(D_ref), axis=-1) > 1e-12 * np.max(np.abs(D_ref))      # rows far above the skip level
        ok = (C_ref[0] * C_ref[1] > 0) & big[0] & big[1]
        if ok.any():
            e_auto, e_te = cl_err(C[c][:, ok], C_ref[:, ok])
            assert e_auto <= TOL_CL and e_te <= TOL_CL
    plan.close()
