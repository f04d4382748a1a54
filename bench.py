#!/usr/bin/env python
"""bench.py -- one JSON line for the line-of-sight hot path.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--impl reference]

A step = one pass of the whole hot path over one batch of seeded synthetic sources that is already
resident in HBM: gcamb_los_transfer + gcamb_los_cls for a single cosmology; at config 3 (64
cosmologies, one plan) gcamb_los_spectra_batched, the fused kernel that shares the j_l recurrence
across the cosmologies of a block and accumulates Eq. 1 without writing Delta (the two-kernel
batched path is timed beside it).
Default workload: BASELINE.json config 1 ("CAMB-default-scale", l = 2..2500), the config the
metric is quoted on.  `value` = nominal (l,k,tau) terms per second = N_l N_k N_tau B per step /
device time per step (reading R19); the executed-term rate (terms not skipped by R16), spectra/s
and the FP64 roofline of the transfer kernel are reported beside it.

N > 1 (torchrun): every rank runs its own cosmology of the same grid (independent problems, no
data-path collective: DESIGN.md "Multi-GPU"), `value` = all ranks' terms / max-over-ranks time.

`--impl reference` times the CPU oracle (oracle/, test infrastructure) on the host cores on a
bounded k-sample of the same workload; there is no reference implementation to install.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2509_25110_b200 import synth  # noqa: E402  (generator only: none of the method's arithmetic)

METRIC = "LOS (l,k,tau) terms/s at lmax=2500"
UNIT = "terms/s"
# FP64 roofline denominator: 148 SMs x 64 DFMA lanes x 2 flop x 1.965 GHz
FP64_LANES_PER_SM = 64
L2_FLUSH_BYTES = 256 << 20
# dram__bytes_read.sum + dram__bytes_write.sum of the transfer call of ONE step (config 3: the fused call), summed over
# its launches, from the committed ncu --set full captures (profiles/r2_kernels.md)
NCU_TRAFFIC_BYTES = {
    0: 5.308e6,
    1: (155.7e6 + 91.24e6) + 3.062e6,
    2: (1.466e9 + 1.327e9) + (0.09813e9 + 0.04122e9),
    3: (5.604e9 + 2.034e9) + (0.5681e9 + 0.007168e9),
    4: (3.948e9 + 4.605e9) + (0.4554e9 + 0.7074e9),
}

def host_cores() -> int:
    try:
        return len(os.sched_getaffinity(0))
    except AttributeError:  # pragma: no cover
        return os.cpu_count() or 1


def workload_config(cfg) -> dict:
    return {
        "workload": f"config {cfg.index} ({cfg.name}): l={cfg.l_min}..{cfg.l_max} (all), n_k={cfg.n_k} log in "
                    f"[{cfg.k_lo:g},{cfg.k_hi:g}], n_tau={cfg.n_tau} ({cfg.n_tau_uniform} uniform + "
                    f"{cfg.n_tau_log} log), sources T,E{',phi' if cfg.with_phi else ''}, batch={cfg.n_batch}",
        "n_l": cfg.n_l, "n_k": cfg.n_k, "n_tau": cfg.n_tau, "n_src": cfg.n_src, "batch": cfg.n_batch,
        "seed": cfg.seed,
    }


# --------------------------------------------------------------------------- clocks
class ClockSampler:
    """Samples SM clock and clock-event reasons through NVML (what nvidia-smi reads) in a thread."""

    REASONS = {
        0x8: "hw_slowdown", 0x40: "hw_thermal_slowdown", 0x20: "sw_thermal_slowdown",
        0x4: "sw_power_cap", 0x80: "hw_power_brake", 0x2: "applications_clocks_setting",
        0x100: "display_clock_setting", 0x10: "sync_boost",
    }

    def __init__(self, torch_device_index: int, period_s: float = 0.001):
        self.period = period_s
        self.samples: list[int] = []
        self.reason_bits = 0
        self.sm_max = None
        self._stop = threading.Event()
        self._thread = None
        self._h = None
        try:
            import pynvml
            import torch
            pynvml.nvmlInit()
            self._nv = pynvml
            uuid = getattr(torch.cuda.get_device_properties(torch_device_index), "uuid", None)
            try:
                self._h = pynvml.nvmlDeviceGetHandleByUUID(f"GPU-{uuid}".encode())
            except Exception:
                self._h = pynvml.nvmlDeviceGetHandleByIndex(torch_device_index)
            self.sm_max = int(pynvml.nvmlDeviceGetMaxClockInfo(self._h, pynvml.NVML_CLOCK_SM))
        except Exception as e:  # NVML missing: report that instead of inventing clocks
            self.error = repr(e)

    def _run(self):
        nv = self._nv
        while not self._stop.is_set():
            try:
                self.samples.append(int(nv.nvmlDeviceGetClockInfo(self._h, nv.NVML_CLOCK_SM)))
                try:
                    bits = nv.nvmlDeviceGetCurrentClocksEventReasons(self._h)
                except Exception:
                    bits = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self._h)
                self.reason_bits |= int(bits)
            except Exception:
                pass
            self._stop.wait(self.period)

    def start(self):
        if self._h is not None:
            self._thread = threading.Thread(target=self._run, daemon=True)
            self._thread.start()

    def stop(self) -> dict:
        self._stop.set()
        if self._thread is not None:
            self._thread.join()
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.sm_max, "reasons": [], "samples": 0,
                    "error": getattr(self, "error", "no samples")}
        reasons = [name for bit, name in self.REASONS.items() if self.reason_bits & bit]
        return {"sm_mhz": float(np.median(self.samples)), "sm_min_mhz": int(min(self.samples)),
                "sm_max_mhz": self.sm_max, "reasons": reasons, "samples": len(self.samples)}


# --------------------------------------------------------------------------- multi-rank bookkeeping
def max_over_ranks(times, dist, device):
    """Element-wise maximum of a list of per-rank times over all ranks (the slowest rank decides)."""
    import torch
    tt = torch.tensor(list(times), dtype=torch.float64, device=device)
    if dist is not None:
        dist.all_reduce(tt, op=dist.ReduceOp.MAX)
    return [float(v) for v in tt.cpu()]


def whole_job_rate(units_per_rank: float, world: int, t_max: float) -> float:
    """Weak scaling over independent replicas: all ranks' units / the slowest rank's time."""
    return units_per_rank * world / t_max


# --------------------------------------------------------------------------- reference arm
def oracle_sample_run(cfg, stride: int, cores: int):
    """The oracle as it stands (fp64 build, OpenMP over k) on every `stride`-th k row of the workload."""
    import oracle
    sl = slice(0, cfg.n_k, stride)
    sl_k = cfg.k()[sl]
    S_T, S_E, S_P = synth.sources(cfg, 0, sl)
    P = synth.primordial_power(cfg, 0)[sl]
    t0 = time.perf_counter()
    D = oracle.transfer(cfg.l_list(), sl_k, cfg.tau(), cfg.tau0, S_T, S_E, S_P, real="f64", nthreads=cores)
    C = oracle.cls(sl_k, D, P, real="f64", nthreads=cores)
    dt = time.perf_counter() - t0
    return dt, D, C, np.arange(cfg.n_k)[sl]


def calibrate_stride(cfg, cores: int, budget_s: float) -> int:
    """k stride whose sample costs about `budget_s` of oracle time (every cost class of the
    ragged workload stays represented: the rows are evenly strided over the log-spaced k grid)."""
    probe = max(1, cfg.n_k // max(2 * cores, 16))
    dt, _, _, rows = oracle_sample_run(cfg, probe, cores)
    per_row = dt / rows.size
    n_rows = max(2, min(cfg.n_k, int(budget_s / max(per_row, 1e-9))))
    return max(1, -(-cfg.n_k // n_rows))


def run_reference(args) -> None:
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    oracle.build()
    cfg = synth.CONFIGS[args.config]
    cores = host_cores()
    budget = min(20.0, 150.0 / max(1, args.steps + args.warmup))
    stride = calibrate_stride(cfg, cores, budget)
    for _ in range(args.warmup):
        oracle_sample_run(cfg, stride, cores)
    runs = [oracle_sample_run(cfg, stride, cores) for _ in range(args.steps)]
    t = float(np.mean([r[0] for r in runs]))
    n_rows = runs[0][3].size
    terms = cfg.n_l * n_rows * cfg.n_tau
    value = terms / t
    sample = f"every {stride}-th k row ({n_rows} of {cfg.n_k}), all l, all tau, one cosmology per step"
    out = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * t, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": workload_config(cfg),
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(out), flush=True)


# --------------------------------------------------------------------------- CUDA arm
def run_cuda(args) -> None:
    import torch

    from paper_2509_25110_b200 import los

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback; --impl reference times the oracle)")
    los.load_library()
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    cfg = synth.CONFIGS[args.config]
    B = cfg.n_batch
    batched = B > 1
    props = torch.cuda.get_device_properties(dev)
    n_sm = props.multi_processor_count

    # ---- inputs: pinned host copies (for the e2e leg) and device-resident copies (for `value`)
    first_c = rank * B
    hS = [[], [], []]
    for c in range(first_c, first_c + B):
        s = synth.sources(cfg, c)
        for q in range(cfg.n_src):
            hS[q].append(s[q])
    hS = [torch.from_numpy(np.stack(x)).pin_memory() if x else None for x in hS]
    hP = torch.from_numpy(np.stack([synth.primordial_power(cfg, c) for c in range(first_c, first_c + B)])).pin_memory()
    dS = [None if x is None else (x.to(dev) if batched else x[0].to(dev)) for x in hS]
    dP = hP.to(dev) if batched else hP[0].to(dev)

    t0 = time.perf_counter()
    plan = los.Plan(cfg.l_list(), cfg.k(), cfg.tau(), cfg.tau0, with_phi=cfg.with_phi)
    torch.cuda.synchronize()
    plan_ms = 1e3 * (time.perf_counter() - t0)

    lead = (B,) if batched else ()
    Delta = torch.empty(lead + (plan.n_src, plan.n_l, plan.n_k), dtype=torch.float64, device=dev)
    Cl = torch.empty(lead + (plan.n_spec, plan.n_l), dtype=torch.float64, device=dev)
    flush = torch.empty(L2_FLUSH_BYTES, dtype=torch.uint8, device=dev)

    fused_info = plan.gcamb_los_spectra_batched_info(B) if batched else {"fused": False}
    fused = fused_info["fused"]

    def transfer_two_kernel():
        if batched:
            plan.gcamb_los_transfer_batched(dS[0], dS[1], dS[2], out=Delta)
        else:
            plan.gcamb_los_transfer(dS[0], dS[1], dS[2], out=Delta)

    def cls_two_kernel():
        if batched:
            plan.gcamb_los_cls_batched(Delta, dP, out=Cl)
        else:
            plan.gcamb_los_cls(Delta, dP, out=Cl)

    if fused:
        # sources -> C_l in one call (fused kernel + finishing kernel); the "cls" leg is empty
        def transfer():
            plan.gcamb_los_spectra_batched(dS[0], dS[1], dS[2], dP, out=Cl)

        def cls():
            pass
        launches_per_step = fused_info["kernels"]
    else:
        transfer, cls = transfer_two_kernel, cls_two_kernel
        launches_per_step = plan.launches_per_step

    for _ in range(args.warmup):
        flush.zero_()
        transfer()
        cls()
    ev = [[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(args.steps)]
    sampler = ClockSampler(local_rank)
    barrier()
    sampler.start()
    wall0 = time.perf_counter()
    for s in range(args.steps):
        flush.zero_()                      # > L2 (126 MB): every step starts with a cold L2
        ev[s][0].record()
        transfer()
        ev[s][1].record()
        cls()
        ev[s][2].record()
    barrier()
    wall = time.perf_counter() - wall0
    clocks = sampler.stop()
    t_transfer = np.array([e[0].elapsed_time(e[1]) for e in ev]) * 1e-3
    t_cls = np.array([e[1].elapsed_time(e[2]) for e in ev]) * 1e-3
    t_step = float(np.mean(t_transfer + t_cls))

    two_kernel = None
    if fused:   # the same batch through gcamb_los_transfer_batched + gcamb_los_cls_batched, for comparison
        n2 = max(3, min(args.steps, 10))
        ev2 = [[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(n2)]
        transfer_two_kernel()
        cls_two_kernel()
        for s in range(n2):
            flush.zero_()
            ev2[s][0].record()
            transfer_two_kernel()
            ev2[s][1].record()
            cls_two_kernel()
            ev2[s][2].record()
        torch.cuda.synchronize()
        Cl_two = Cl.clone()
        transfer()
        torch.cuda.synchronize()
        two_kernel = {
            "transfer_ms": float(np.mean([e[0].elapsed_time(e[1]) for e in ev2])),
            "cls_ms": float(np.mean([e[1].elapsed_time(e[2]) for e in ev2])),
            "max_rel_diff_TT_EE": float(((Cl[:, :2] - Cl_two[:, :2]).abs() / Cl_two[:, :2].abs()).max()),
        }
        two_kernel["spectra_per_s"] = B / ((two_kernel["transfer_ms"] + two_kernel["cls_ms"]) * 1e-3)

    # ---- e2e: the public host-buffer call, H2D of the sources and D2H of C_l inside the timed region
    hCl = torch.empty((B, plan.n_spec, plan.n_l), dtype=torch.float64).pin_memory()
    e2e_steps = max(3, min(args.steps, 20))
    for _ in range(2):
        plan.gcamb_los_spectra_host(hS[0], hS[1], hS[2], hP, hCl)
    barrier()
    e0 = time.perf_counter()
    for _ in range(e2e_steps):
        plan.gcamb_los_spectra_host(hS[0], hS[1], hS[2], hP, hCl)   # synchronises its stream
    torch.cuda.synchronize()
    t_e2e = (time.perf_counter() - e0) / e2e_steps
    barrier()
    if fused:   # the host entry point runs the two-kernel path: same sums in another order
        same = bool(np.allclose(hCl.numpy().reshape(Cl.shape), Cl.cpu().numpy(), rtol=1e-9, atol=0.0))
    else:
        same = bool(np.array_equal(hCl.numpy().reshape(Cl.shape), Cl.cpu().numpy()))
    h2d = sum(int(x.numel()) * 8 for x in hS if x is not None) + int(hP.numel()) * 8
    d2h = int(hCl.numel()) * 8

    # ---- max over ranks
    t_step, t_e2e, t_tr, t_cl = max_over_ranks(
        [t_step, t_e2e, float(np.mean(t_transfer)), float(np.mean(t_cls))], dist, dev)

    nominal = plan.nominal_terms * B
    executed = plan.executed_terms * B
    if fused:
        # a block of BC cosmologies shares the coefficient and the recurrence: 2 + n_src BC FP64 lane-slots
        # per (l, k, tau) for BC cosmologies; executed counts (l, k, tau, cosmology)
        bc = 8 if (B > 4 and plan.n_tau <= 1280) else 4
        flop_per_term = 2 * (2 + plan.n_src * bc) / bc
        kernel_name = "fused_kernel"
        algorithmic = (f"{flop_per_term} flop per executed (l,k,tau,cosmology): (2 + {plan.n_src} x {bc}) FP64 FMA lane-slots "
                       f"per (l,k,tau) shared by a block of {bc} cosmologies, x {executed} executed terms per launch; "
                       f"the time is that of the whole call (fused kernel + finishing kernel)")
    else:
        flop_per_term = 2 * (2 + plan.n_src)         # coefficient + recurrence + n_src accumulate DFMAs
        kernel_name = "transfer_kernel"
        algorithmic = f"{flop_per_term} flop per executed term x {executed} executed terms per launch"
    peak_tf = n_sm * FP64_LANES_PER_SM * 2 * (clocks.get("sm_max_mhz") or 1965.0) * 1e6 / 1e12
    achieved_tf = executed * flop_per_term / t_tr / 1e12

    # measured FP64 ceilings of this device, same process (libgcamb_probe.so, not part of the method):
    # dependent DFMA chains (8 per thread) and mma.sync.m8n8k4.f64 chains (8 per warp, 256 FMA each)
    probe_out = torch.empty(n_sm * 8 * 256, dtype=torch.float64, device=dev)
    iters = 1 << 14

    def probe_tflops(fn, fma_per_thread_iter):
        fn(n_sm * 8, 256, iters, probe_out)
        p0, p1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        p0.record()
        fn(n_sm * 8, 256, iters, probe_out)
        p1.record()
        torch.cuda.synchronize()
        return n_sm * 8 * 256 * fma_per_thread_iter * iters * 2 / (p0.elapsed_time(p1) * 1e-3) / 1e12

    probe_tf = probe_tflops(los.gcamb_probe_dfma, 8)
    probe_dmma_tf = probe_tflops(los.gcamb_probe_dmma, 8 * 256 / 32)

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    out = {
        "metric": METRIC, "value": whole_job_rate(nominal, world, t_step), "unit": UNIT, "n_gpus": world,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * t_step,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic",
        "config": {**workload_config(cfg), "l2": f"flushed between steps ({L2_FLUSH_BYTES >> 20} MiB memset)",
                   "per_rank": "one cosmology batch per GPU, no collective on the data path"},
        "executed_terms_per_s": executed * world / t_step,
        "executed_fraction": plan.executed_terms / plan.nominal_terms,
        "spectra_per_s": B * world / t_step,
        "transfer_ms": 1e3 * t_tr, "cls_ms": 1e3 * t_cl, "plan_create_ms": plan_ms,
        "wall_ms_per_step_incl_flush": 1e3 * wall / args.steps,
        "clocks": clocks,
        **({"two_kernel_path": two_kernel} if two_kernel else {}),
        "e2e": {"value": nominal * world / t_e2e, "unit": UNIT, "h2d_bytes_per_step": h2d,
                "d2h_bytes_per_step": d2h, "ms_per_step": 1e3 * t_e2e, "api": "gcamb_los_spectra_host",
                "matches_device_path": same},
        "gpu_launches": launches_per_step * args.steps,
        "roofline": {
            "bound": "alu", "kernel": kernel_name, "achieved": achieved_tf, "peak": peak_tf,
            "unit": "TFLOP/s", "frac": achieved_tf / peak_tf, "traffic": NCU_TRAFFIC_BYTES.get(args.config),
            "traffic_unit": "bytes per transfer call (ncu dram read+write of its launches, profiles/r2_kernels.md)",
            "peak_source": f"derived: {n_sm} SMs x {FP64_LANES_PER_SM} DFMA/clk x 2 x sm_max_mhz (DESIGN.md); "
                           f"dfma probe measured {probe_tf:.2f} TFLOP/s, dmma (m8n8k4.f64) probe "
                           f"{probe_dmma_tf:.2f} TFLOP/s in this process",
            "algorithmic": algorithmic,
            "frac_of_measured_dfma": achieved_tf / probe_tf,
        },
    }

    if world == 1 and not args.no_cpu_baseline:
        import oracle
        oracle.build()
        cores = host_cores()
        stride = calibrate_stride(cfg, cores, 15.0)
        dt, D_ref, _, rows = oracle_sample_run(cfg, stride, cores)
        D_gpu = (Delta[0] if batched else Delta)[:, :, torch.from_numpy(rows).to(dev)].cpu().numpy()
        scale = np.max(np.abs(D_ref), axis=-1, keepdims=True)
        err = float(np.max(np.abs(D_gpu - D_ref) / np.where(scale > 0, scale, 1.0)))
        out["cpu_baseline"] = {
            "value": cfg.n_l * rows.size * cfg.n_tau / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": f"every {stride}-th k row ({rows.size} of {cfg.n_k}), all l, all tau, cosmology 0; "
                      f"fp64 oracle build, {dt:.1f} s",
            "delta_err_on_sample": err,
        }
    print(json.dumps(out), flush=True)
    plan.close()
    if dist is not None:
        dist.destroy_process_group()


# --------------------------------------------------------------------------- SURVEY 8(f) "next" rows
def camb_like_l_list(l_min: int, l_max: int) -> np.ndarray:
    """Every l below 40, every 10th to 200, every 50th above (CAMB's default sampling)."""
    l = np.concatenate([np.arange(l_min, 40), np.arange(40, 200, 10), np.arange(200, l_max + 1, 50), [l_max]])
    return np.unique(l[(l >= l_min) & (l <= l_max)]).astype(np.int32)


def tensor_sources(k: np.ndarray, tau: np.ndarray, seed: int = synth.SEED):
    """Seeded synthetic tensor sources (the recipe of tests/test_gpu_tensor.py)."""
    kk, tt = k[:, None], tau[None, :]
    g = np.exp(-((tt - 280.0) ** 2) / (2.0 * 20.0 ** 2)) / (20.0 * np.sqrt(2.0 * np.pi))
    damp = np.exp(-((kk / 0.05) ** 2))
    h = np.sin(kk * tt) / (kk * tt)
    S = [g * h * damp + 0.3e-4 * np.exp(-(((tt - 10000.0) / 2500.0) ** 2)) * np.exp(-kk / 0.005),
         g * h * damp * 0.2, g * np.cos(kk * tt) * damp * 0.15]
    return [np.ascontiguousarray(x * (1.0 + 1e-3 * synth.uniform_pm1(seed, 500 + q, 0, x.size).reshape(x.shape)))
            for q, x in enumerate(S)]


def time_steps(step_fns, steps: int, warmup: int, flush):
    """Mean CUDA-event time (ms) of each function of a step, L2 flushed before every step."""
    import torch
    for _ in range(warmup):
        flush.zero_()
        for f in step_fns:
            f()
    ev = [[torch.cuda.Event(enable_timing=True) for _ in range(len(step_fns) + 1)] for _ in range(steps)]
    for s in range(steps):
        flush.zero_()
        ev[s][0].record()
        for i, f in enumerate(step_fns):
            f()
            ev[s][i + 1].record()
    torch.cuda.synchronize()
    return [float(np.mean([e[i].elapsed_time(e[i + 1]) for e in ev])) for i in range(len(step_fns))]


def run_next(args) -> None:
    """One JSON line for a SURVEY 8(f) row: --workload sparse | tensor | open | srcinterp | emulator (single GPU)."""
    import torch

    import oracle
    from paper_2509_25110_b200 import los

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback)")
    los.load_library()
    torch.cuda.set_device(0)
    dev = torch.device("cuda", 0)
    n_sm = torch.cuda.get_device_properties(dev).multi_processor_count
    cfg = synth.CONFIGS[1]
    tau, tau0 = cfg.tau(), cfg.tau0
    flush = torch.empty(L2_FLUSH_BYTES, dtype=torch.uint8, device=dev)
    to_dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(dev)
    cores = host_cores()
    oracle.build()
    w = args.workload
    sampler = ClockSampler(0)
    sampler.start()
    extra = {}
    if w == "sparse":      # NEXT-2: CAMB's default operating mode on config-1 grids
        k, l_list = cfg.k(), camb_like_l_list(cfg.l_min, cfg.l_max)
        S = synth.sources(cfg)
        plan = los.Plan(l_list, k, tau, tau0)
        dS, dP = [to_dev(S[0]), to_dev(S[1])], to_dev(synth.primordial_power(cfg))
        D = torch.empty((2, plan.n_l, plan.n_k), dtype=torch.float64, device=dev)
        C = torch.empty((3, plan.n_l), dtype=torch.float64, device=dev)
        C_all = torch.empty((3, plan.n_l_all), dtype=torch.float64, device=dev)
        fns = [lambda: plan.gcamb_los_transfer(dS[0], dS[1], out=D), lambda: plan.gcamb_los_cls(D, dP, out=C),
               lambda: plan.gcamb_los_cl_interp(C, out=C_all)]
        names = ["transfer_ms", "cls_ms", "cl_interp_ms"]
        tiles = np.unique((cfg.l_max - l_list) // 8).size / ((cfg.l_max - cfg.l_min) // 8 + 1)
        flop_per_term = 2 * (2 + 2 * tiles)       # recurrence everywhere, accumulates on the tiles that hold a listed l
        units = plan.n_l_all * plan.n_k * plan.n_tau
        workload = (f"config-1 grids, CAMB-like list of {l_list.size} of {plan.n_l_all} multipoles: sparse transfer + cls + "
                    f"spline to every l (reading R25)")
        algorithmic = (f"{flop_per_term:.3f} flop per walked (l,k,tau): coefficient + recurrence on every l, 2 accumulates on "
                       f"the {100 * tiles:.0f} % of l-tiles that hold a listed l")
        ref = lambda sl: oracle.transfer(l_list, k[sl], tau, tau0, S[0][sl], S[1][sl], real="f64", nthreads=cores)
        get_rows = lambda rows: D[:, :, rows]
    elif w == "tensor":    # NEXT-3: l_max_tensor = 1500, k tau0 <= 3000, config-1 tau grid
        k, l_list = synth.k_grid(1000, 1e-5, 3000.0 / tau0), np.arange(2, 1501, dtype=np.int32)
        S = tensor_sources(k, tau)
        plan = los.Plan(l_list, k, tau, tau0, tensor=True)
        dS, dP = [to_dev(x) for x in S], to_dev(2.1e-10 * (k / 0.05) ** -0.01)
        D = torch.empty((3, plan.n_l, plan.n_k), dtype=torch.float64, device=dev)
        C = torch.empty((4, plan.n_l), dtype=torch.float64, device=dev)
        work = torch.empty(plan.gcamb_los_tensor_work_bytes() // 8, dtype=torch.float64, device=dev)
        fns = [lambda: plan.gcamb_los_transfer_tensor(*dS, out=D, work=work), lambda: plan.gcamb_los_cls_tensor(D, dP, out=C)]
        names = ["transfer_ms", "cls_ms"]
        flop_per_term, units = 2 * 6, plan.n_l * plan.n_k * plan.n_tau
        workload = "tensor modes: l=2..1500, n_k=1000 log in [1e-5, 3000/tau0], config-1 tau grid (1200), sources T,E,B (reading R27)"
        algorithmic = ("12 flop per executed (l,k,tau): coefficient + recurrence + the 4 plain sums the T, E, B kernels reduce to "
                       "(the sums with one power of 1/x follow from those without through j_l/x = (j_{l-1} + j_{l+1})/(2l+1)); "
                       "one walk of the four-sum transfer kernels executes exactly those")
        ref = lambda sl: oracle.transfer_tensor(l_list, k[sl], tau, tau0, S[0][sl], S[1][sl], S[2][sl], real="f64", nthreads=cores)
        get_rows = lambda rows: D[:, :, rows]
    elif w == "open":      # NEXT-4: config-1 grids in an open universe, r_c = 14000 Mpc
        k, l_list, K = cfg.k(), cfg.l_list(), -1.0 / 14000.0 ** 2
        S = synth.sources(cfg)
        plan = los.Plan(l_list, k, tau, tau0, curvature_K=K)
        dS, dP = [to_dev(S[0]), to_dev(S[1])], to_dev(synth.primordial_power(cfg))
        D = torch.empty((2, plan.n_l, plan.n_k), dtype=torch.float64, device=dev)
        C = torch.empty((3, plan.n_l), dtype=torch.float64, device=dev)
        fns = [lambda: plan.gcamb_los_transfer(dS[0], dS[1], out=D), lambda: plan.gcamb_los_cls(D, dP, out=C)]
        names = ["transfer_ms", "cls_ms"]
        flop_per_term, units = 2 * 5, plan.n_l * plan.n_k * plan.n_tau
        workload = "config-1 grids in an open universe, K = -1/(14000 Mpc)^2: hyperspherical Bessel functions (reading R28)"
        algorithmic = "10 flop per executed (l,k,tau): A_l coth, R_l f_{l+1}, recurrence, 2 accumulates"
        ref = lambda sl: oracle.transfer_open(l_list, k[sl], tau, tau0, K, S[0][sl], S[1][sl], real="f64", nthreads=cores)
        get_rows = lambda rows: D[:, :, rows]
    elif w == "emulator":  # NEXT-1 + NEXT-2: the batch of config 3 on CAMB's default l sampling, fused kernel + spline to every l
        cfg3 = synth.CONFIGS[3]
        B = cfg3.n_batch
        k, l_list = cfg3.k(), camb_like_l_list(cfg3.l_min, cfg3.l_max)
        S0 = synth.sources(cfg3, 0)
        dT = torch.empty((B, cfg3.n_k, cfg3.n_tau), dtype=torch.float64, device=dev)
        dE = torch.empty_like(dT)
        hP = np.stack([synth.primordial_power(cfg3, c) for c in range(B)])
        for c in range(B):
            Sc_ = S0 if c == 0 else synth.sources(cfg3, c)
            dT[c].copy_(torch.from_numpy(Sc_[0])); dE[c].copy_(torch.from_numpy(Sc_[1]))
        dP = to_dev(hP)
        plan = los.Plan(l_list, k, tau, tau0)
        info = plan.gcamb_los_spectra_batched_info(B)
        C = torch.empty((B, 3, plan.n_l), dtype=torch.float64, device=dev)
        C_all = torch.empty((B, 3, plan.n_l_all), dtype=torch.float64, device=dev)
        fns = [lambda: plan.gcamb_los_spectra_batched(dT, dE, None, dP, out=C), lambda: plan.gcamb_los_cl_interp(C, out=C_all)]
        names = ["spectra_batched_ms", "cl_interp_ms"]
        # algorithmic work: coefficient + recurrence once per executed (l, k, tau) for a block of 8 cosmologies, two
        # accumulates per cosmology on the LISTED l only; the listed share of the executed terms, exactly
        x = k[:, None] * (tau0 - tau)[None, :]
        L = np.minimum(np.ceil(x + 18.2 * np.cbrt(x) + 8.0), cfg3.l_max)          # reading R16
        n_exec = np.maximum(L - cfg3.l_min + 1, 0.0)
        n_listed = np.searchsorted(l_list, L, side="right").astype(np.float64)
        f_listed = float(n_listed.sum() / n_exec.sum())
        workload = (f"config 3 batch ({B} cosmologies, config-1 grids) on a CAMB-like list of {l_list.size} of {plan.n_l_all} "
                    f"multipoles: gcamb_los_spectra_batched ({'fused kernel' if info['fused'] else 'two kernels'}) + spline to every l")
    else:                  # srcinterp, NEXT-3: 300 evolved wavenumbers -> the 3000 of config 1, T and E
        k, kc = cfg.k(), synth.k_grid(300, cfg.k_lo, cfg.k_hi)
        coarse = synth.Config(9, "coarse", cfg.l_min, cfg.l_max, 300, cfg.k_lo, cfg.k_hi, cfg.n_tau_uniform, cfg.n_tau_log, False)
        Sc = np.stack(synth.sources(coarse, noise=False)[:2])
        plan = los.Plan(np.arange(2, 10, dtype=np.int32), k, tau, tau0)
        si = los.SourceInterp(plan, kc)
        dSc = to_dev(Sc)
        out = torch.empty((2, plan.n_k, plan.n_tau), dtype=torch.float64, device=dev)
        work = torch.empty_like(dSc)
        fns = [lambda: si.gcamb_los_interp_sources(dSc, out=out, work=work)]
        names = ["interp_sources_ms"]
        workload = "InterpolateSources: 300 coarse -> 3000 fine wavenumbers of config 1, 1200 tau, sources T and E (reading R26)"
    times = time_steps(fns, args.steps, args.warmup, flush)
    clocks = sampler.stop()
    t_step = sum(times) * 1e-3
    peak_tf = n_sm * FP64_LANES_PER_SM * 2 * (clocks.get("sm_max_mhz") or 1965.0) * 1e6 / 1e12
    if w == "emulator":
        executed = plan.executed_terms
        flop = 2.0 * (2.0 / 8.0 + 2.0 * f_listed)
        achieved = executed * B * flop / (times[0] * 1e-3) / 1e12
        value, unit, metric = plan.n_l_all * plan.n_k * plan.n_tau * B / t_step, UNIT, "LOS (l,k,tau) terms/s"
        roof = {"bound": "alu", "kernel": "fused_kernel", "achieved": achieved, "peak": peak_tf, "unit": "TFLOP/s",
                "frac": achieved / peak_tf, "traffic": None,
                "peak_source": f"derived: {n_sm} SMs x {FP64_LANES_PER_SM} DFMA/clk x 2 x sm_max_mhz (DESIGN.md section 7)",
                "algorithmic": (f"{flop:.3f} flop per executed (l,k,tau,cosmology): coefficient + recurrence shared by 8 cosmologies, 2 "
                                f"accumulates on the {100 * f_listed:.1f} % of the executed terms whose l is listed; x {executed} executed "
                                f"terms x {B} cosmologies; the kernel accumulates whole l-tiles of 8 (every tile that holds a listed l)")}
        extra = {"executed_terms_per_s": executed * B / t_step, "spectra_per_s": B / t_step, "fused": bool(info["fused"])}
        t0 = time.perf_counter()
        D_ref = oracle.transfer(l_list, k, tau, tau0, S0[0], S0[1], real="f64", nthreads=cores)
        C_ref = oracle.cl_interp(l_list, oracle.cls(k, D_ref, hP[0], real="f64"), real="f64")
        dt = time.perf_counter() - t0
        got = C_all[0].cpu().numpy()
        err = float(max(np.max(np.abs(got[:2] / C_ref[:2] - 1.0)),
                        np.max(np.abs(got[2] - C_ref[2]) / np.sqrt(C_ref[2] ** 2 + C_ref[0] * C_ref[1]))))
        cpu = {"value": 1.0 / dt, "unit": "spectra/s", "cores": cores, "kind": "oracle",
               "sample": f"cosmology 0 in full (sparse transfer + cls + spline), fp64 oracle build, {dt:.1f} s", "cl_err_on_sample": err}
    elif w == "srcinterp":
        # algorithmic bytes: coarse sources read once, second derivatives written and read once, fine sources written
        n_c, n_f = int(dSc.numel()), int(out.numel())
        bytes_alg = 8 * (3 * n_c + n_f)
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json"))) if os.path.exists(os.path.join(ROOT, "MEASURED_PEAKS.json")) else {}
        peak_gbs = float(peaks.get("hbm_gbs", 6650.0))
        value, unit, metric = n_f / t_step, "source values/s", "interpolated source values/s (InterpolateSources)"
        roof = {"bound": "hbm", "kernel": "srcinterp_mma_kernel + srcinterp_eval_kernel", "achieved": bytes_alg / t_step / 1e9,
                "peak": peak_gbs, "unit": "GB/s", "frac": bytes_alg / t_step / 1e9 / peak_gbs, "traffic": None,
                "peak_source": "MEASURED_PEAKS.json hbm_gbs" if peaks else "fallback 6650 GB/s (B200_PROFILING.md)",
                "algorithmic": f"{bytes_alg} bytes per call: 8 (3 n_coarse + n_fine) n_tau n_series"}
        t0 = time.perf_counter()
        ref_out = oracle.interp_sources(kc, k, Sc[0], real="f64")
        dt = time.perf_counter() - t0
        err = float(np.max(np.abs(out[0].cpu().numpy() - ref_out)) / np.max(np.abs(Sc[0])))
        cpu = {"value": ref_out.size / dt, "unit": unit, "cores": 1, "kind": "oracle",
               "sample": f"source T in full (one of two series), fp64 oracle build, {dt:.2f} s", "err_on_sample": err}
        si.close()
    else:
        executed = plan.executed_terms
        value, unit, metric = units / t_step, UNIT, "LOS (l,k,tau) terms/s"
        achieved = executed * flop_per_term / (times[0] * 1e-3) / 1e12
        roof = {"bound": "alu", "kernel": "transfer_kernel", "achieved": achieved, "peak": peak_tf, "unit": "TFLOP/s",
                "frac": achieved / peak_tf, "traffic": None,
                "peak_source": f"derived: {n_sm} SMs x {FP64_LANES_PER_SM} DFMA/clk x 2 x sm_max_mhz (DESIGN.md section 7)",
                "algorithmic": f"{algorithmic}, x {executed} executed terms per call; time = the transfer call"}
        extra = {"executed_terms_per_s": executed / t_step, "spectra_per_s": 1.0 / t_step}
        if w == "tensor":
            # the same transfer call for a batch of 4 cosmologies (gcamb_los_transfer_tensor_batched): a single call is 1000
            # thread blocks at two per SM, whose heaviest row is 3/4 of an SM's share; a batch fills the tail
            Bt = 4
            dSb = [x.unsqueeze(0).repeat(Bt, 1, 1).contiguous() for x in dS]
            Db = torch.empty((Bt,) + tuple(D.shape), dtype=torch.float64, device=dev)
            workb = torch.empty(Bt * (plan.gcamb_los_tensor_work_bytes() // 8), dtype=torch.float64, device=dev)
            tb = time_steps([lambda: plan.gcamb_los_transfer_tensor_batched(*dSb, out=Db, work=workb)], min(args.steps, 20), 3, flush)
            extra["batched"] = {"n_batch": Bt, "transfer_ms_per_cosmology": tb[0] / Bt,
                                "roofline_frac": executed * flop_per_term / (tb[0] / Bt * 1e-3) / 1e12 / peak_tf,
                                "equals_single_call": bool(torch.equal(Db[Bt - 1], D))}
        # a bounded k sample (about 10 s of oracle time), evenly strided so that every cost class is represented
        stride = max(1, k.size // max(2 * cores, 16))
        t0 = time.perf_counter()
        ref(slice(0, k.size, stride))
        per_row = (time.perf_counter() - t0) / len(range(0, k.size, stride))
        stride = max(1, -(-k.size // max(2, min(k.size, int(10.0 / max(per_row, 1e-9))))))
        sl = slice(0, k.size, stride)
        t0 = time.perf_counter()
        D_ref = ref(sl)
        dt = time.perf_counter() - t0
        rows = np.arange(k.size)[sl]
        D_gpu = get_rows(torch.from_numpy(rows).to(dev)).cpu().numpy()
        scale = np.max(np.abs(D_ref), axis=-1, keepdims=True)
        err = float(np.max(np.abs(D_gpu - D_ref) / np.where(scale > 0, scale, 1.0)))
        cpu = {"value": units / k.size * rows.size / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
               "sample": f"every {stride}-th k row ({rows.size} of {k.size}), fp64 oracle build, {dt:.1f} s",
               "delta_err_on_sample": err}
    out_line = {
        "metric": metric, "value": value, "unit": unit, "n_gpus": 1, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": 1e3 * t_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic", "config": {"workload": workload, "l2": f"flushed between steps ({L2_FLUSH_BYTES >> 20} MiB memset)"},
        **{n: t for n, t in zip(names, times)}, **extra, "clocks": clocks, "roofline": roof, "cpu_baseline": cpu,
    }
    print(json.dumps(out_line), flush=True)
    plan.close()


def main() -> None:
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=None)
    ap.add_argument("--warmup", type=int, default=None)
    ap.add_argument("--config", type=int, default=1, choices=range(len(synth.CONFIGS)))
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--workload", default="config", choices=["config", "sparse", "tensor", "open", "srcinterp", "emulator"],
                    help="config: BASELINE.json's configs (--config); the others: SURVEY 8(f) rows, one GPU")
    args = ap.parse_args()
    if args.workload != "config":
        if args.impl != "cuda" or args.gpus != 1:
            raise SystemExit("bench.py: --workload rows run on one GPU with the CUDA arm only")
        args.steps = 50 if args.steps is None else args.steps
        args.warmup = 5 if args.warmup is None else max(args.warmup, 3)
        run_next(args)
    elif args.impl == "reference":
        args.steps = 3 if args.steps is None else args.steps
        args.warmup = 1 if args.warmup is None else args.warmup
        run_reference(args)
    else:
        args.steps = 100 if args.steps is None else args.steps
        args.warmup = 5 if args.warmup is None else max(args.warmup, 3)
        run_cuda(args)


if __name__ == "__main__":
    main()
