"""Thin ctypes binding of libgcamb_los.so (include/gcamb_los.h): argument marshalling only.

Every step of the path runs in the CUDA kernels behind the C ABI; torch is used for device
memory and streams.  There is no CPU fallback: if the library is missing or no CUDA device is
present the calls raise.
"""
from __future__ import annotations

import ctypes
import os

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libgcamb_los.so")

GCAMB_SRC_T, GCAMB_SRC_E, GCAMB_SRC_PHI, GCAMB_SRC_TENSOR = 1, 2, 4, 8
_STATUS = {0: "GCAMB_OK", 1: "GCAMB_EINVAL", 2: "GCAMB_EGRID", 3: "GCAMB_EALLOC", 4: "GCAMB_ECUDA"}

EXPORTS = (
    "gcamb_los_plan_create", "gcamb_los_plan_create_curved", "gcamb_los_plan_destroy", "gcamb_los_plan_info", "gcamb_los_plan_launches",
    "gcamb_los_transfer",
    "gcamb_los_cls", "gcamb_los_transfer_batched", "gcamb_los_cls_batched", "gcamb_los_spectra_host",
    "gcamb_los_spectra_batched", "gcamb_los_spectra_batched_info", "gcamb_los_cl_interp", "gcamb_los_last_error",
    "gcamb_los_tensor_work_bytes", "gcamb_los_transfer_tensor", "gcamb_los_cls_tensor",
    "gcamb_los_transfer_tensor_batched", "gcamb_los_cls_tensor_batched",
    "gcamb_los_srcinterp_create", "gcamb_los_srcinterp_destroy", "gcamb_los_srcinterp_info", "gcamb_los_interp_sources",
    "gcamb_los_interp_sources_noalloc",
)
# libgcamb_probe.so (include/gcamb_probe.h): bench.py's roofline probes, not part of the method
PROBE_LIB_PATH = os.path.join(_HERE, "libgcamb_probe.so")
PROBE_EXPORTS = ("gcamb_probe_dfma", "gcamb_probe_dmma")

_vp, _i32, _i64, _f64 = ctypes.c_void_p, ctypes.c_int32, ctypes.c_int64, ctypes.c_double
_lib = None


class GcambError(RuntimeError):
    def __init__(self, status: int, message: str):
        super().__init__(f"{_STATUS.get(status, status)}: {message}")
        self.status = status


def load_library() -> ctypes.CDLL:
    """dlopen the in-tree library; fails loudly if it has not been built."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} not built: run `python -m paper_2509_25110_b200.build` "
                          "(there is no CPU fallback)")
    lib = ctypes.CDLL(LIB_PATH)
    lib.gcamb_los_last_error.restype = ctypes.c_char_p
    lib.gcamb_los_plan_create.argtypes = [ctypes.POINTER(_vp), _vp, _i32, _vp, _i32, _vp, _i32, _f64,
                                          ctypes.c_uint32, _vp]
    lib.gcamb_los_plan_create_curved.argtypes = [ctypes.POINTER(_vp), _vp, _i32, _vp, _i32, _vp, _i32, _f64, _f64,
                                               ctypes.c_uint32, _vp]
    lib.gcamb_los_plan_destroy.argtypes = [_vp]
    lib.gcamb_los_plan_info.argtypes = [_vp] + [ctypes.POINTER(_i32)] * 5 + [ctypes.POINTER(_i64)]
    lib.gcamb_los_plan_launches.argtypes = [_vp, ctypes.POINTER(_i32), ctypes.POINTER(_i32)]
    lib.gcamb_los_transfer.argtypes = [_vp, _vp, _vp, _vp, _vp, _vp]
    lib.gcamb_los_cls.argtypes = [_vp, _vp, _vp, _vp, _vp]
    lib.gcamb_los_transfer_batched.argtypes = [_vp, _i32, _vp, _vp, _vp, _vp, _vp]
    lib.gcamb_los_cls_batched.argtypes = [_vp, _i32, _vp, _vp, _vp, _vp]
    lib.gcamb_los_spectra_host.argtypes = [_vp, _i32, _vp, _vp, _vp, _vp, _vp, _vp, _vp]
    lib.gcamb_los_spectra_batched.argtypes = [_vp, _i32, _vp, _vp, _vp, _vp, _vp, _vp]
    lib.gcamb_los_spectra_batched_info.argtypes = [_vp, _i32, ctypes.POINTER(_i32), ctypes.POINTER(_i32),
                                                   ctypes.POINTER(_i64)]
    lib.gcamb_los_cl_interp.argtypes = [_vp, _i32, _vp, _vp, _vp]
    lib.gcamb_los_tensor_work_bytes.argtypes = [_vp, ctypes.POINTER(_i64)]
    lib.gcamb_los_transfer_tensor.argtypes = [_vp, _vp, _vp, _vp, _vp, _vp, _vp]
    lib.gcamb_los_cls_tensor.argtypes = [_vp, _vp, _vp, _vp, _vp]
    lib.gcamb_los_transfer_tensor_batched.argtypes = [_vp, _i32, _vp, _vp, _vp, _vp, _vp, _vp]
    lib.gcamb_los_cls_tensor_batched.argtypes = [_vp, _i32, _vp, _vp, _vp, _vp]
    lib.gcamb_los_srcinterp_create.argtypes = [ctypes.POINTER(_vp), _vp, _vp, _i32, _vp]
    lib.gcamb_los_srcinterp_destroy.argtypes = [_vp]
    lib.gcamb_los_srcinterp_info.argtypes = [_vp] + [ctypes.POINTER(_i32)] * 4
    lib.gcamb_los_interp_sources.argtypes = [_vp, _i32, _vp, _vp, _vp, _vp]
    lib.gcamb_los_interp_sources_noalloc.argtypes = [_vp, _i32, _vp, _vp, _vp]
    _lib = lib
    return lib


def _check(status: int) -> None:
    if status != 0:
        raise GcambError(status, load_library().gcamb_los_last_error().decode())


def _stream() -> int:
    return torch.cuda.current_stream().cuda_stream


def _dev(t: torch.Tensor | None, shape, name: str) -> int | None:
    if t is None:
        return None
    if not (t.is_cuda and t.dtype == torch.float64 and t.is_contiguous()):
        raise TypeError(f"{name}: need a contiguous float64 CUDA tensor")
    if tuple(t.shape) != tuple(shape):
        raise ValueError(f"{name}: shape {tuple(t.shape)} != {tuple(shape)}")
    return t.data_ptr()


def _host(a, shape, name: str) -> np.ndarray | None:
    if a is None:
        return None
    if isinstance(a, torch.Tensor):
        a = a.numpy()
    if not (isinstance(a, np.ndarray) and a.dtype == np.float64 and a.flags.c_contiguous):
        raise TypeError(f"{name}: need a C-contiguous float64 host array")
    if tuple(a.shape) != tuple(shape):
        raise ValueError(f"{name}: shape {tuple(a.shape)} != {tuple(shape)}")
    return a


class Plan:
    """gcamb_los_plan: grids, quadrature weights and recurrence start values on the device."""

    def __init__(self, l_list, k, tau, tau0: float, with_phi: bool = False, tensor: bool = False,
                 curvature_K: float = 0.0):
        if not torch.cuda.is_available():
            raise RuntimeError("gcamb_los needs a CUDA device (no CPU fallback)")
        lib = load_library()
        l_list = np.ascontiguousarray(l_list, dtype=np.int32)
        k = np.ascontiguousarray(k, dtype=np.float64)
        tau = np.ascontiguousarray(tau, dtype=np.float64)
        mask = GCAMB_SRC_TENSOR if tensor else GCAMB_SRC_T | GCAMB_SRC_E | (GCAMB_SRC_PHI if with_phi else 0)
        self.tensor = bool(tensor)
        handle = _vp()
        if curvature_K != 0.0:      # K < 0 open, K > 0 closed universe
            _check(lib.gcamb_los_plan_create_curved(ctypes.byref(handle), l_list.ctypes.data, l_list.size,
                                                  k.ctypes.data, k.size, tau.ctypes.data, tau.size,
                                                  float(tau0), float(curvature_K), mask, _stream()))
        else:
            _check(lib.gcamb_los_plan_create(ctypes.byref(handle), l_list.ctypes.data, l_list.size,
                                             k.ctypes.data, k.size, tau.ctypes.data, tau.size,
                                             float(tau0), mask, _stream()))
        self._h = handle
        out = [_i32() for _ in range(5)]
        ex = _i64()
        _check(lib.gcamb_los_plan_info(self._h, *[ctypes.byref(o) for o in out], ctypes.byref(ex)))
        self.n_l, self.n_k, self.n_tau, self.n_src, self.n_spec = (o.value for o in out)
        self.n_l_all = int(l_list[-1] - l_list[0] + 1)      # integer multipoles spanned by the l list
        self.executed_terms = ex.value
        self.nominal_terms = self.n_l * self.n_k * self.n_tau
        # kernels of this library one transfer + one cls call launch (bench.py's gpu_launches)
        nt, nc = _i32(), _i32()
        _check(lib.gcamb_los_plan_launches(self._h, ctypes.byref(nt), ctypes.byref(nc)))
        self.transfer_launches, self.cls_launches = nt.value, nc.value
        self.launches_per_step = nt.value + nc.value

    def close(self) -> None:
        if getattr(self, "_h", None):
            _check(load_library().gcamb_los_plan_destroy(self._h))
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- device-resident calls (asynchronous on torch's current stream)
    def gcamb_los_transfer(self, S_T, S_E, S_phi=None, out=None) -> torch.Tensor:
        return self.gcamb_los_transfer_batched(S_T, S_E, S_phi, out, _batched=False)

    def gcamb_los_transfer_batched(self, S_T, S_E, S_phi=None, out=None, _batched=True) -> torch.Tensor:
        B = (S_T.shape[0],) if _batched else ()
        sh = B + (self.n_k, self.n_tau)
        if out is None:
            out = torch.empty(B + (self.n_src, self.n_l, self.n_k), dtype=torch.float64, device=S_T.device)
        pT, pE, pP = _dev(S_T, sh, "S_T"), _dev(S_E, sh, "S_E"), _dev(S_phi, sh, "S_phi")
        pD = _dev(out, B + (self.n_src, self.n_l, self.n_k), "Delta")
        lib = load_library()
        if _batched:
            _check(lib.gcamb_los_transfer_batched(self._h, B[0], pT, pE, pP, pD, _stream()))
        else:
            _check(lib.gcamb_los_transfer(self._h, pT, pE, pP, pD, _stream()))
        return out

    def gcamb_los_cls(self, Delta, P_R, out=None) -> torch.Tensor:
        return self.gcamb_los_cls_batched(Delta, P_R, out, _batched=False)

    def gcamb_los_cls_batched(self, Delta, P_R, out=None, _batched=True) -> torch.Tensor:
        B = (Delta.shape[0],) if _batched else ()
        if out is None:
            out = torch.empty(B + (self.n_spec, self.n_l), dtype=torch.float64, device=Delta.device)
        pD = _dev(Delta, B + (self.n_src, self.n_l, self.n_k), "Delta")
        pP = _dev(P_R, B + (self.n_k,), "P_R")
        pC = _dev(out, B + (self.n_spec, self.n_l), "Cl")
        lib = load_library()
        if _batched:
            _check(lib.gcamb_los_cls_batched(self._h, B[0], pD, pP, pC, _stream()))
        else:
            _check(lib.gcamb_los_cls(self._h, pD, pP, pC, _stream()))
        return out

    # ---- tensor modes (plans created with tensor=True)
    def gcamb_los_tensor_work_bytes(self) -> int:
        n = _i64()
        _check(load_library().gcamb_los_tensor_work_bytes(self._h, ctypes.byref(n)))
        return n.value

    def gcamb_los_transfer_tensor(self, S_T, S_E, S_B, out=None, work=None) -> torch.Tensor:
        """Tensor sources [n_k][n_tau] x 3 -> Delta [3][n_l][n_k] (T, E, B)."""
        sh = (self.n_k, self.n_tau)
        if out is None:
            out = torch.empty((3, self.n_l, self.n_k), dtype=torch.float64, device=S_T.device)
        n_work = self.gcamb_los_tensor_work_bytes() // 8
        if work is None:
            work = torch.empty(n_work, dtype=torch.float64, device=S_T.device)
        _check(load_library().gcamb_los_transfer_tensor(
            self._h, _dev(S_T, sh, "S_T"), _dev(S_E, sh, "S_E"), _dev(S_B, sh, "S_B"),
            _dev(out, (3, self.n_l, self.n_k), "Delta"), _dev(work, (n_work,), "work"), _stream()))
        return out

    def gcamb_los_cls_tensor(self, Delta, P_t, out=None) -> torch.Tensor:
        """Delta [3][n_l][n_k] -> C_l [4][n_l] (TT, EE, BB, TE)."""
        if out is None:
            out = torch.empty((4, self.n_l), dtype=torch.float64, device=Delta.device)
        _check(load_library().gcamb_los_cls_tensor(
            self._h, _dev(Delta, (3, self.n_l, self.n_k), "Delta"), _dev(P_t, (self.n_k,), "P_t"),
            _dev(out, (4, self.n_l), "Cl"), _stream()))
        return out

    def gcamb_los_transfer_tensor_batched(self, S_T, S_E, S_B, out=None, work=None) -> torch.Tensor:
        """Tensor sources [B][n_k][n_tau] x 3 -> Delta [B][3][n_l][n_k]; scratch of B x gcamb_los_tensor_work_bytes()."""
        B = S_T.shape[0]
        sh = (B, self.n_k, self.n_tau)
        if out is None:
            out = torch.empty((B, 3, self.n_l, self.n_k), dtype=torch.float64, device=S_T.device)
        n_work = B * (self.gcamb_los_tensor_work_bytes() // 8)
        if work is None:
            work = torch.empty(n_work, dtype=torch.float64, device=S_T.device)
        _check(load_library().gcamb_los_transfer_tensor_batched(
            self._h, B, _dev(S_T, sh, "S_T"), _dev(S_E, sh, "S_E"), _dev(S_B, sh, "S_B"),
            _dev(out, (B, 3, self.n_l, self.n_k), "Delta"), _dev(work, (n_work,), "work"), _stream()))
        return out

    def gcamb_los_cls_tensor_batched(self, Delta, P_t, out=None) -> torch.Tensor:
        """Delta [B][3][n_l][n_k], P_t [B][n_k] -> C_l [B][4][n_l] (TT, EE, BB, TE)."""
        B = Delta.shape[0]
        if out is None:
            out = torch.empty((B, 4, self.n_l), dtype=torch.float64, device=Delta.device)
        _check(load_library().gcamb_los_cls_tensor_batched(
            self._h, B, _dev(Delta, (B, 3, self.n_l, self.n_k), "Delta"), _dev(P_t, (B, self.n_k), "P_t"),
            _dev(out, (B, 4, self.n_l), "Cl"), _stream()))
        return out

    def gcamb_los_cl_interp(self, Cl, out=None) -> torch.Tensor:
        """C_l on the l list [..., n_spec, n_l] -> C_l on every integer l [..., n_spec, l_last - l_first + 1]."""
        lead = tuple(Cl.shape[:-2])
        n_batch = int(np.prod(lead)) if lead else 1
        if out is None:
            out = torch.empty(lead + (self.n_spec, self.n_l_all), dtype=torch.float64, device=Cl.device)
        _check(load_library().gcamb_los_cl_interp(
            self._h, n_batch, _dev(Cl, lead + (self.n_spec, self.n_l), "Cl"),
            _dev(out, lead + (self.n_spec, self.n_l_all), "Cl_all"), _stream()))
        return out

    def gcamb_los_spectra_batched(self, S_T, S_E, S_phi, P_R, out=None) -> torch.Tensor:
        """Sources of a batch -> C_l [B][n_spec][n_l] (fused kernel when the plan allows it)."""
        B = S_T.shape[0]
        sh = (B, self.n_k, self.n_tau)
        if out is None:
            out = torch.empty((B, self.n_spec, self.n_l), dtype=torch.float64, device=S_T.device)
        _check(load_library().gcamb_los_spectra_batched(
            self._h, B, _dev(S_T, sh, "S_T"), _dev(S_E, sh, "S_E"), _dev(S_phi, sh, "S_phi"),
            _dev(P_R, (B, self.n_k), "P_R"), _dev(out, (B, self.n_spec, self.n_l), "Cl"), _stream()))
        return out

    def gcamb_los_spectra_batched_info(self, n_batch: int) -> dict:
        fused, kernels, scratch = _i32(), _i32(), _i64()
        _check(load_library().gcamb_los_spectra_batched_info(self._h, n_batch, ctypes.byref(fused),
                                                             ctypes.byref(kernels), ctypes.byref(scratch)))
        return {"fused": bool(fused.value), "kernels": kernels.value, "scratch_bytes": scratch.value}

    # ---- host buffers in, host buffers out (H2D + kernels + D2H inside the call)
    def gcamb_los_spectra_host(self, S_T, S_E, S_phi, P_R, Cl_out, Delta_out=None) -> None:
        B = S_T.shape[0]
        sh = (B, self.n_k, self.n_tau)
        aT, aE, aP = _host(S_T, sh, "S_T"), _host(S_E, sh, "S_E"), _host(S_phi, sh, "S_phi")
        aR = _host(P_R, (B, self.n_k), "P_R")
        aC = _host(Cl_out, (B, self.n_spec, self.n_l), "Cl")
        aD = _host(Delta_out, (B, self.n_src, self.n_l, self.n_k), "Delta")
        _check(load_library().gcamb_los_spectra_host(
            self._h, B, aT.ctypes.data, aE.ctypes.data, None if aP is None else aP.ctypes.data,
            aR.ctypes.data, aC.ctypes.data, None if aD is None else aD.ctypes.data, _stream()))


def gcamb_los_plan_create(l_list, k, tau, tau0, with_phi=False, tensor=False) -> Plan:
    return Plan(l_list, k, tau, tau0, with_phi, tensor)


class SourceInterp:
    """gcamb_los_srcinterp: sources on a coarse k grid -> sources on the plan's k grid (InterpolateSources)."""

    def __init__(self, plan: Plan, k_coarse):
        k_coarse = np.ascontiguousarray(k_coarse, dtype=np.float64)
        handle = _vp()
        _check(load_library().gcamb_los_srcinterp_create(ctypes.byref(handle), plan._h, k_coarse.ctypes.data,
                                                         k_coarse.size, _stream()))
        self._h = handle
        self.n_kc, self.n_k, self.n_tau = int(k_coarse.size), plan.n_k, plan.n_tau
        band = _i32()
        _check(load_library().gcamb_los_srcinterp_info(self._h, None, None, None, ctypes.byref(band)))
        self.band_columns = band.value          # 0: the solve runs as sequential sweeps

    def close(self) -> None:
        if getattr(self, "_h", None):
            _check(load_library().gcamb_los_srcinterp_destroy(self._h))
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def gcamb_los_interp_sources(self, S_coarse, out=None, work=None) -> torch.Tensor:
        """[..., n_kc, n_tau] -> [..., n_k, n_tau]; the leading dimensions are independent series."""
        lead = tuple(S_coarse.shape[:-2])
        n_series = int(np.prod(lead)) if lead else 1
        if out is None:
            out = torch.empty(lead + (self.n_k, self.n_tau), dtype=torch.float64, device=S_coarse.device)
        if work is None:
            work = torch.empty_like(S_coarse)
        _check(load_library().gcamb_los_interp_sources(
            self._h, n_series, _dev(S_coarse, lead + (self.n_kc, self.n_tau), "S_coarse"),
            _dev(out, lead + (self.n_k, self.n_tau), "S_fine"), _dev(work, lead + (self.n_kc, self.n_tau), "work"),
            _stream()))
        return out

    def gcamb_los_interp_sources_noalloc(self, S_coarse, out) -> torch.Tensor:
        """As gcamb_los_interp_sources, with the library's static device scratch (at most 2^20 doubles of coarse
        sources): the call allocates nothing, so `out` is the caller's."""
        lead = tuple(S_coarse.shape[:-2])
        n_series = int(np.prod(lead)) if lead else 1
        _check(load_library().gcamb_los_interp_sources_noalloc(
            self._h, n_series, _dev(S_coarse, lead + (self.n_kc, self.n_tau), "S_coarse"),
            _dev(out, lead + (self.n_k, self.n_tau), "S_fine"), _stream()))
        return out


_probe_lib = None


def load_probe_library() -> ctypes.CDLL:
    global _probe_lib
    if _probe_lib is None:
        if not os.path.exists(PROBE_LIB_PATH):
            raise ImportError(f"{PROBE_LIB_PATH} not built: run `python -m paper_2509_25110_b200.build`")
        lib = ctypes.CDLL(PROBE_LIB_PATH)
        for name in PROBE_EXPORTS:
            getattr(lib, name).argtypes = [_i32, _i32, _i64, _vp, _vp]
        _probe_lib = lib
    return _probe_lib


def _probe(name: str, blocks: int, threads: int, iters: int, out: torch.Tensor) -> None:
    rc = getattr(load_probe_library(), name)(blocks, threads, iters, _dev(out, (blocks * threads,), "out"), _stream())
    if rc:
        raise RuntimeError(f"{name}: cudaError {rc}")


def gcamb_probe_dfma(blocks: int, threads: int, iters: int, out: torch.Tensor) -> None:
    _probe("gcamb_probe_dfma", blocks, threads, iters, out)


def gcamb_probe_dmma(blocks: int, threads: int, iters: int, out: torch.Tensor) -> None:
    _probe("gcamb_probe_dmma", blocks, threads, iters, out)
