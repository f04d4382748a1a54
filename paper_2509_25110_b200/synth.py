"""Seeded synthetic inputs for the line-of-sight path (grids, sources, P_R, noise).

This module is the ONE piece shared by the CUDA path's tests/bench and the CPU oracle's
tests. It holds none of the method's arithmetic (no Bessel functions, no quadrature
weights, no transfer or C_l sums): it only writes the arrays both sides read.

The paper's workloads are CAMB source functions for Planck LCDM (Sec. 3.1);
CAMB is not available, so BASELINE.json's analytic source model stands in for them
(DESIGN.md "Input recipe"). Readings R7-R11 and R22 of SURVEY.md Sec. 8(c) fix every detail:

  k grid   k_j = a (b/a)^(j/(N-1)), j = 0..N-1                                   (R7)
  tau grid n_u uniform points on [200, 400] (both ends) followed by n_log points
           tau = 400 (tau_end/400)^(m/n_log), m = 1..n_log, tau_end = tau0 - 1   (R8)
  g(tau)   normalised Gaussian pdf N(mu, sigma)                                   (R9)
  S_T      g cos(c_s k tau) exp(-(k/0.1)^2) + 2 exp(-((tau-11000)/2000)^2) exp(-k/0.01)
  S_E      g k sin(c_s k tau) exp(-(k/0.1)^2)
  S_phi    exp(-((tau-9000)/3000)^2) k^-2 exp(-k/0.2)
  noise    S <- S (1 + 1e-3 u), u in [-1, 1) from a counter-based splitmix64     (R10)
  P_R      A_s (k/0.05)^(n_s-1)                                                   (R11)
  config 3 per-cosmology draws of sigma, mu, c_s, A_s, n_s                        (R22)
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

TAU0 = 14000.0
SEED = 1234
_GOLDEN = np.uint64(0x9E3779B97F4A7C15)
_STREAM_MULT = 0xD1342543DE82EF95
_MASK = (1 << 64) - 1


# --------------------------------------------------------------------------- noise
def _mix_int(v: int) -> int:
    """One splitmix64 output for state v (python ints, mod 2^64)."""
    z = (v + 0x9E3779B97F4A7C15) & _MASK
    z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & _MASK
    z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & _MASK
    return z ^ (z >> 31)


def _mix_np(v: np.ndarray) -> np.ndarray:
    with np.errstate(over="ignore"):
        z = v + _GOLDEN
        z = (z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
        z = (z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
        return z ^ (z >> np.uint64(31))


def stream_base(seed: int, stream: int) -> int:
    return _mix_int((seed + stream * _STREAM_MULT) & _MASK)


def uniform_pm1(seed: int, stream: int, start: int, count: int) -> np.ndarray:
    """u_n in [-1, 1) for n = start .. start+count-1 of (seed, stream)."""
    base = np.uint64(stream_base(seed, stream))
    with np.errstate(over="ignore"):
        n = np.arange(start, start + count, dtype=np.uint64) + base
    z = _mix_np(n)
    return (z >> np.uint64(11)).astype(np.float64) * 2.0 ** -52 - 1.0


# --------------------------------------------------------------------------- grids
def k_grid(n_k: int, k_lo: float, k_hi: float) -> np.ndarray:
    j = np.arange(n_k, dtype=np.float64)
    k = k_lo * (k_hi / k_lo) ** (j / (n_k - 1))
    k[0], k[-1] = k_lo, k_hi
    return k


def tau_grid(n_uniform: int, n_log: int, tau0: float = TAU0) -> np.ndarray:
    tau_end = tau0 - 1.0
    i = np.arange(n_uniform, dtype=np.float64)
    tu = 200.0 + 200.0 * i / (n_uniform - 1)
    tu[-1] = 400.0
    m = np.arange(1, n_log + 1, dtype=np.float64)
    tl = 400.0 * (tau_end / 400.0) ** (m / n_log)
    tl[-1] = tau_end
    return np.concatenate([tu, tl])


# --------------------------------------------------------------------------- configs
@dataclass(frozen=True)
class Config:
    """One of BASELINE.json's five configs (zero-based)."""
    index: int
    name: str
    l_min: int
    l_max: int
    n_k: int
    k_lo: float
    k_hi: float
    n_tau_uniform: int
    n_tau_log: int
    with_phi: bool
    n_batch: int = 1
    tau0: float = TAU0
    seed: int = SEED

    @property
    def n_tau(self) -> int:
        return self.n_tau_uniform + self.n_tau_log

    @property
    def n_l(self) -> int:
        return self.l_max - self.l_min + 1

    @property
    def n_src(self) -> int:
        return 3 if self.with_phi else 2

    @property
    def n_spec(self) -> int:
        return 4 if self.with_phi else 3

    def l_list(self) -> np.ndarray:
        return np.arange(self.l_min, self.l_max + 1, dtype=np.int32)

    def k(self) -> np.ndarray:
        return k_grid(self.n_k, self.k_lo, self.k_hi)

    def tau(self) -> np.ndarray:
        return tau_grid(self.n_tau_uniform, self.n_tau_log, self.tau0)

    def nominal_terms(self) -> int:
        return self.n_batch * self.n_l * self.n_k * self.n_tau


CONFIGS = (
    Config(0, "tiny", 2, 200, 400, 1e-4, 0.3, 200, 100, False),
    Config(1, "camb-default-scale", 2, 2500, 3000, 1e-5, 0.6, 600, 600, False),
    Config(2, "high-accuracy", 2, 6000, 10000, 1e-5, 1.0, 1500, 1500, True),
    Config(3, "emulator-batch", 2, 2500, 3000, 1e-5, 0.6, 600, 600, False, n_batch=64),
    Config(4, "extreme", 2, 10000, 20000, 1e-5, 1.2, 2000, 2000, True),
)


@dataclass(frozen=True)
class Cosmology:
    """Per-cosmology parameters of the analytic source model (R9, R11, R22)."""
    sigma: float = 20.0
    mu: float = 280.0
    c_s: float = 1.0 / np.sqrt(3.0)
    A_s: float = 2.1e-9
    n_s: float = 0.965


def cosmology(cfg: Config, c: int) -> Cosmology:
    """Cosmology c of a config: fixed fiducial except for the emulator batch (R22)."""
    if cfg.n_batch == 1:
        return Cosmology()
    u = 0.5 * (uniform_pm1(cfg.seed, 1000 + c, 0, 5) + 1.0)  # U[0,1)
    return Cosmology(
        sigma=15.0 + 10.0 * u[0],
        mu=260.0 + 40.0 * u[1],
        c_s=0.55 + 0.05 * u[2],
        A_s=(1.9 + 0.4 * u[3]) * 1e-9,
        n_s=0.94 + 0.05 * u[4],
    )


# --------------------------------------------------------------------------- sources
def _noise(seed: int, stream: int, n_k: int, n_tau: int, k_slice: slice) -> np.ndarray:
    j0, j1, step = k_slice.indices(n_k)
    assert step > 0
    u = uniform_pm1(seed, stream, j0 * n_tau, max(j1 - j0, 0) * n_tau)
    return 1.0 + 1e-3 * u.reshape(max(j1 - j0, 0), n_tau)[::step]


def sources(cfg: Config, c: int = 0, k_slice: slice = slice(None), noise: bool = True):
    """S_T, S_E, (S_phi or None) as [n_k_slice][n_tau] float64, tau fastest, for cosmology c.

    `k_slice` selects rows of the k grid; noise indices follow the FULL grid
    (n = j*N_tau + i), so a slice reproduces the same values as the full array.
    """
    cos = cosmology(cfg, c)
    k = cfg.k()[k_slice][:, None]
    tau = cfg.tau()[None, :]
    g = np.exp(-((tau - cos.mu) ** 2) / (2.0 * cos.sigma ** 2)) / (cos.sigma * np.sqrt(2.0 * np.pi))
    damp = np.exp(-((k / 0.1) ** 2))
    late = 2.0 * np.exp(-(((tau - 11000.0) / 2000.0) ** 2)) * np.exp(-k / 0.01)
    S_T = g * np.cos(cos.c_s * k * tau) * damp + late
    S_E = g * k * np.sin(cos.c_s * k * tau) * damp
    S_phi = None
    if cfg.with_phi:
        S_phi = np.exp(-(((tau - 9000.0) / 3000.0) ** 2)) * k ** -2.0 * np.exp(-k / 0.2)
        S_phi = np.ascontiguousarray(np.broadcast_to(S_phi, S_T.shape))
    if noise:
        S_T = S_T * _noise(cfg.seed, 3 * c + 0, cfg.n_k, cfg.n_tau, k_slice)
        S_E = S_E * _noise(cfg.seed, 3 * c + 1, cfg.n_k, cfg.n_tau, k_slice)
        if S_phi is not None:
            S_phi = S_phi * _noise(cfg.seed, 3 * c + 2, cfg.n_k, cfg.n_tau, k_slice)
    return np.ascontiguousarray(S_T), np.ascontiguousarray(S_E), S_phi


def primordial_power(cfg: Config, c: int = 0) -> np.ndarray:
    """P_R(k_j) = A_s (k/0.05)^(n_s-1)  (R11)."""
    cos = cosmology(cfg, c)
    return cos.A_s * (cfg.k() / 0.05) ** (cos.n_s - 1.0)
