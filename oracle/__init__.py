"""ctypes access to the CPU oracle (oracle/los_oracle.c).

TEST INFRASTRUCTURE ONLY: imported by tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs; never by paper_2509_25110_b200/.  Two builds of the same
C file: `f64` (REAL = double, the fp64 oracle and the timed CPU baseline) and `f80`
(REAL = x87 long double, the grading reference of reading R14).
"""
from __future__ import annotations

import ctypes
import os
import subprocess
import threading

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "los_oracle.c")
_FLAGS = ["-O2", "-std=c11", "-fno-fast-math", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared"]
_LOCK = threading.Lock()
_LIBS: dict[str, ctypes.CDLL] = {}

_pd = ctypes.POINTER(ctypes.c_double)
_pi = ctypes.POINTER(ctypes.c_int32)


def lib_path(real: str) -> str:
    return os.path.join(_HERE, f"liblos_oracle_{real}.so")


def build(force: bool = False) -> None:
    """Compile both oracle builds with gcc (a few seconds)."""
    for real, defs in (("f64", []), ("f80", ["-DORACLE_LONG_DOUBLE"])):
        out = lib_path(real)
        if not force and os.path.exists(out) and os.path.getmtime(out) >= os.path.getmtime(_SRC):
            continue
        tmp = f"{out}.{os.getpid()}.tmp"
        subprocess.run(["gcc", *_FLAGS, *defs, _SRC, "-o", tmp, "-lm"], check=True)
        os.replace(tmp, out)


def _lib(real: str) -> ctypes.CDLL:
    if real not in ("f64", "f80"):
        raise ValueError("real must be 'f64' or 'f80'")
    with _LOCK:
        if real not in _LIBS:
            build()
            lib = ctypes.CDLL(lib_path(real))
            lib.oracle_real_mant_bits.restype = ctypes.c_int
            lib.oracle_lcut.argtypes = [ctypes.c_double]
            lib.oracle_lcut.restype = ctypes.c_int
            lib.oracle_sph_bessel.argtypes = [ctypes.c_double, ctypes.c_int, ctypes.c_int, _pd]
            lib.oracle_trapz_weights.argtypes = [_pd, ctypes.c_int, _pd]
            lib.oracle_transfer.argtypes = [_pi, ctypes.c_int, _pd, ctypes.c_int, _pd, ctypes.c_int,
                                            ctypes.c_double, _pd, _pd, _pd, ctypes.c_int, ctypes.c_int, _pd]
            lib.oracle_cls.argtypes = [ctypes.c_int, ctypes.c_int, _pd, ctypes.c_int, _pd, _pd,
                                       ctypes.c_int, _pd]
            lib.oracle_cl_interp.argtypes = [_pi, ctypes.c_int, ctypes.c_int, _pd, _pd]
            lib.oracle_sph_bessel_derivs.argtypes = [ctypes.c_double, ctypes.c_int, ctypes.c_int, _pd]
            lib.oracle_transfer_tensor.argtypes = [_pi, ctypes.c_int, _pd, ctypes.c_int, _pd, ctypes.c_int,
                                                   ctypes.c_double, _pd, _pd, _pd, ctypes.c_int, ctypes.c_int, _pd]
            lib.oracle_cls_tensor.argtypes = [ctypes.c_int, _pd, ctypes.c_int, _pd, _pd, ctypes.c_int, _pd]
            lib.oracle_hyp_lcut_open.argtypes = [ctypes.c_double, ctypes.c_double]
            lib.oracle_hyp_lcut_open.restype = ctypes.c_int
            lib.oracle_hyp_lcut_closed.argtypes = [ctypes.c_double, ctypes.c_double]
            lib.oracle_hyp_lcut_closed.restype = ctypes.c_int
            lib.oracle_hyp_bessel_closed.argtypes = [ctypes.c_double, ctypes.c_double, ctypes.c_int, ctypes.c_int, _pd]
            lib.oracle_transfer_closed.argtypes = [_pi, ctypes.c_int, _pd, ctypes.c_int, _pd, ctypes.c_int,
                                                   ctypes.c_double, ctypes.c_double, _pd, _pd, _pd, ctypes.c_int,
                                                   ctypes.c_int, _pd]
            lib.oracle_hyp_bessel_open.argtypes = [ctypes.c_double, ctypes.c_double, ctypes.c_int, ctypes.c_int, _pd]
            lib.oracle_transfer_open.argtypes = [_pi, ctypes.c_int, _pd, ctypes.c_int, _pd, ctypes.c_int,
                                                 ctypes.c_double, ctypes.c_double, _pd, _pd, _pd, ctypes.c_int,
                                                 ctypes.c_int, _pd]
            lib.oracle_interp_sources.argtypes = [_pd, ctypes.c_int, _pd, ctypes.c_int, ctypes.c_int, _pd, _pd]
            assert lib.oracle_real_mant_bits() == (53 if real == "f64" else 64)
            _LIBS[real] = lib
        return _LIBS[real]


def _f64(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.float64)


def _ptr(a: np.ndarray):
    return a.ctypes.data_as(_pd)


DEFAULT_MARGIN = 30


def lcut(x: float) -> int:
    return _lib("f64").oracle_lcut(float(x))


def sph_bessel(x: float, lmax: int, margin: int = DEFAULT_MARGIN, real: str = "f64") -> np.ndarray:
    """j_l(x), l = 0..lmax."""
    out = np.empty(lmax + 1, dtype=np.float64)
    if _lib(real).oracle_sph_bessel(float(x), int(lmax), int(margin), _ptr(out)):
        raise ValueError("oracle_sph_bessel: bad arguments")
    return out


def trapz_weights(t, real: str = "f64") -> np.ndarray:
    t = _f64(t)
    w = np.empty_like(t)
    if _lib(real).oracle_trapz_weights(_ptr(t), t.size, _ptr(w)):
        raise ValueError("oracle_trapz_weights: bad arguments")
    return w


def transfer(l_list, k, tau, tau0, S_T, S_E, S_phi=None, margin: int = DEFAULT_MARGIN,
             real: str = "f64", nthreads: int = 0) -> np.ndarray:
    """Delta[n_src][n_l][n_k] (Eq. 2-3)."""
    l_list = np.ascontiguousarray(l_list, dtype=np.int32)
    k, tau, S_T, S_E = _f64(k), _f64(tau), _f64(S_T), _f64(S_E)
    assert S_T.shape == (k.size, tau.size) and S_E.shape == S_T.shape
    sp = None
    if S_phi is not None:
        S_phi = _f64(S_phi)
        assert S_phi.shape == S_T.shape
        sp = _ptr(S_phi)
    n_src = 3 if S_phi is not None else 2
    out = np.empty((n_src, l_list.size, k.size), dtype=np.float64)
    rc = _lib(real).oracle_transfer(l_list.ctypes.data_as(_pi), l_list.size, _ptr(k), k.size,
                                    _ptr(tau), tau.size, float(tau0), _ptr(S_T), _ptr(S_E), sp,
                                    int(margin), int(nthreads), _ptr(out))
    if rc:
        raise ValueError(f"oracle_transfer failed ({rc})")
    return out


def cls(k, Delta, P_R, real: str = "f64", nthreads: int = 0) -> np.ndarray:
    """C_l[n_spec][n_l] (Eq. 1), order TT, EE, TE, (phiphi)."""
    k, Delta, P_R = _f64(k), _f64(Delta), _f64(P_R)
    n_src, n_l, n_k = Delta.shape
    assert n_k == k.size == P_R.size
    out = np.empty((3 if n_src == 2 else 4, n_l), dtype=np.float64)
    rc = _lib(real).oracle_cls(n_src, n_l, _ptr(k), n_k, _ptr(Delta), _ptr(P_R), int(nthreads), _ptr(out))
    if rc:
        raise ValueError(f"oracle_cls failed ({rc})")
    return out


def cl_interp(l_list, Cl_samp, real: str = "f64") -> np.ndarray:
    """C_l on every integer l from l_list[0] to l_list[-1] from C_l on the sparse list (reading R25:
    natural cubic spline of l(l+1) C_l in l).  Cl_samp [n_spec][n_l] -> [n_spec][l_last - l_first + 1]."""
    l_list = np.ascontiguousarray(l_list, dtype=np.int32)
    Cl_samp = _f64(Cl_samp)
    n_spec, n_l = Cl_samp.shape
    assert n_l == l_list.size
    out = np.empty((n_spec, int(l_list[-1] - l_list[0] + 1)), dtype=np.float64)
    rc = _lib(real).oracle_cl_interp(l_list.ctypes.data_as(_pi), n_l, n_spec, _ptr(Cl_samp), _ptr(out))
    if rc:
        raise ValueError(f"oracle_cl_interp failed ({rc})")
    return out


def sph_bessel_derivs(x: float, lmax: int, margin: int = DEFAULT_MARGIN, real: str = "f64") -> np.ndarray:
    """[3][lmax+1]: j_l(x), j_l'(x), j_l''(x), l = 0..lmax (the derivatives are those the tensor kernels use)."""
    out = np.empty((3, lmax + 1), dtype=np.float64)
    if _lib(real).oracle_sph_bessel_derivs(float(x), int(lmax), int(margin), _ptr(out)):
        raise ValueError("oracle_sph_bessel_derivs: bad arguments")
    return out


def transfer_tensor(l_list, k, tau, tau0, S_T, S_E, S_B, margin: int = DEFAULT_MARGIN,
                    real: str = "f64", nthreads: int = 0) -> np.ndarray:
    """Tensor transfer functions Delta[3][n_l][n_k], order T, E, B (reading R27)."""
    l_list = np.ascontiguousarray(l_list, dtype=np.int32)
    k, tau, S_T, S_E, S_B = _f64(k), _f64(tau), _f64(S_T), _f64(S_E), _f64(S_B)
    assert S_T.shape == (k.size, tau.size) and S_E.shape == S_T.shape and S_B.shape == S_T.shape
    out = np.empty((3, l_list.size, k.size), dtype=np.float64)
    rc = _lib(real).oracle_transfer_tensor(l_list.ctypes.data_as(_pi), l_list.size, _ptr(k), k.size,
                                           _ptr(tau), tau.size, float(tau0), _ptr(S_T), _ptr(S_E), _ptr(S_B),
                                           int(margin), int(nthreads), _ptr(out))
    if rc:
        raise ValueError(f"oracle_transfer_tensor failed ({rc})")
    return out


def cls_tensor(k, Delta, P_t, real: str = "f64", nthreads: int = 0) -> np.ndarray:
    """Tensor spectra C_l[4][n_l], order TT, EE, BB, TE (Eq. 1 with P_t, reading R27)."""
    k, Delta, P_t = _f64(k), _f64(Delta), _f64(P_t)
    n_src, n_l, n_k = Delta.shape
    assert n_src == 3 and n_k == k.size == P_t.size
    out = np.empty((4, n_l), dtype=np.float64)
    rc = _lib(real).oracle_cls_tensor(n_l, _ptr(k), n_k, _ptr(Delta), _ptr(P_t), int(nthreads), _ptr(out))
    if rc:
        raise ValueError(f"oracle_cls_tensor failed ({rc})")
    return out


def interp_sources(k_coarse, k, S_coarse, real: str = "f64") -> np.ndarray:
    """Sources on a coarse k grid [n_kc][n_tau] -> sources on k [n_k][n_tau]: natural cubic spline in k for
    every tau (reading R26)."""
    k_coarse, k, S_coarse = _f64(k_coarse), _f64(k), _f64(S_coarse)
    n_kc, n_tau = S_coarse.shape
    assert n_kc == k_coarse.size
    out = np.empty((k.size, n_tau), dtype=np.float64)
    rc = _lib(real).oracle_interp_sources(_ptr(k_coarse), n_kc, _ptr(k), k.size, n_tau, _ptr(S_coarse), _ptr(out))
    if rc:
        raise ValueError(f"oracle_interp_sources failed ({rc})")
    return out


def hyp_lcut_open(beta: float, chi: float) -> int:
    return _lib("f64").oracle_hyp_lcut_open(float(beta), float(chi))


def hyp_bessel_open(beta: float, chi: float, lmax: int, margin: int = DEFAULT_MARGIN, real: str = "f64") -> np.ndarray:
    """Hyperspherical Bessel functions of an open universe Phi_l^beta(chi), l = 0..lmax (reading R28)."""
    out = np.empty(lmax + 1, dtype=np.float64)
    if _lib(real).oracle_hyp_bessel_open(float(beta), float(chi), int(lmax), int(margin), _ptr(out)):
        raise ValueError("oracle_hyp_bessel_open: bad arguments")
    return out


def hyp_lcut_closed(beta: float, chi: float) -> int:
    return _lib("f64").oracle_hyp_lcut_closed(float(beta), float(chi))


def hyp_bessel_closed(beta: float, chi: float, lmax: int, margin: int = DEFAULT_MARGIN, real: str = "f64") -> np.ndarray:
    """Hyperspherical Bessel functions of a closed universe (integer beta >= 3, chi <= pi/2), zero for l >= beta."""
    out = np.empty(lmax + 1, dtype=np.float64)
    if _lib(real).oracle_hyp_bessel_closed(float(beta), float(chi), int(lmax), int(margin), _ptr(out)):
        raise ValueError("oracle_hyp_bessel_closed: bad arguments")
    return out


def transfer_open(l_list, k, tau, tau0, curv_K, S_T, S_E, S_phi=None, margin: int = DEFAULT_MARGIN,
                  real: str = "f64", nthreads: int = 0) -> np.ndarray:
    """Delta[n_src][n_l][n_k] in a curved universe: curv_K < 0 open, > 0 closed (reading R28)."""
    l_list = np.ascontiguousarray(l_list, dtype=np.int32)
    k, tau, S_T, S_E = _f64(k), _f64(tau), _f64(S_T), _f64(S_E)
    assert S_T.shape == (k.size, tau.size) and S_E.shape == S_T.shape
    sp = None
    if S_phi is not None:
        S_phi = _f64(S_phi)
        sp = _ptr(S_phi)
    out = np.empty((3 if S_phi is not None else 2, l_list.size, k.size), dtype=np.float64)
    fn = _lib(real).oracle_transfer_open if curv_K < 0 else _lib(real).oracle_transfer_closed
    rc = fn(l_list.ctypes.data_as(_pi), l_list.size, _ptr(k), k.size, _ptr(tau),
                                         tau.size, float(tau0), float(curv_K), _ptr(S_T), _ptr(S_E), sp,
                                         int(margin), int(nthreads), _ptr(out))
    if rc:
        raise ValueError(f"oracle_transfer_open/closed failed ({rc})")
    return out


transfer_curved = transfer_open      # curv_K < 0: open, curv_K > 0: closed
