"""Seeded synthetic input generators for the SAIL hot path (shared by oracle tests, GPU tests, bench).

This module builds PROBLEM INPUTS only: grids, the correlation data F(tau) of a known
spectrum (Eq. 1 of the paper, by numerical quadrature of the continuous
S(omega)), noise, error bars, sum-rule constants and temperature schedules.  It contains
none of the method's arithmetic (no bin model Eq. 6-8, no move, no chi^2, no branching, no
Philox): it is the only module that both `oracle/` and the CUDA path are fed from, and it
imports neither of them.

Workload recipe = BASELINE.json `configs` with the readings of SURVEY.md §8(c) G4-G10
(restated in DESIGN.md §3):
  * S(omega) = [0.5*0.1/((w-1)^2+0.1^2) + 0.5*0.3/((w-3)^2+0.3^2)] / Z on [0,8], 0 above;
    Z makes int_0^8 S = 1 (atan closed form).
  * omega grid: N_omega uniform bins, LEFT edges omega_k = k*domega on [0, omega_max].
  * tau grid: tau_j = j*dtau, j = 0..N_tau-1 (includes tau = 0, Eq. 2).
  * F_clean(tau) = (1/2pi) int_0^8 S(w) exp(-w tau) dw by composite Simpson, 1e6 intervals.
  * noisy F = F_clean*(1 + eps*xi_j), xi ~ N(0,1) from numpy Philox bit generator (seed);
    sigma_j = eps*F_clean_j.
  * A = F_noisy(0)*2pi/domega (Eq. 16), B = (1/domega) int_0^8 w S dw (closed form).
  * T_s = T0*(T1/T0)^(s/(S-1)), geometric.
These stand in for the paper's workload class (two-peak Lorentzian band, §5.2),
whose actual input files are not available.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

TWO_PI = 2.0 * math.pi

# --- the test spectrum -------------------------------------------------------------------
_PEAKS = ((0.5, 1.0, 0.1), (0.5, 3.0, 0.3))  # (weight, centre, half width)
_SUPPORT = 8.0


def _raw_cdf(w):
    """int_{-inf..w} of the un-normalised double Lorentzian (up to a constant): sum wt*atan((w-w0)/G)."""
    w = np.asarray(w, dtype=np.float64)
    return sum(wt * np.arctan((w - w0) / g) for wt, w0, g in _PEAKS)


def _raw_first_moment_antiderivative(w):
    """Antiderivative of w*S_raw(w): wt*[(G/2) ln((w-w0)^2+G^2) + w0*atan((w-w0)/G)]."""
    w = np.asarray(w, dtype=np.float64)
    return sum(wt * (0.5 * g * np.log((w - w0) ** 2 + g * g) + w0 * np.arctan((w - w0) / g))
               for wt, w0, g in _PEAKS)


Z_RAW = float(_raw_cdf(_SUPPORT) - _raw_cdf(0.0))
FIRST_MOMENT = float((_raw_first_moment_antiderivative(_SUPPORT)
                      - _raw_first_moment_antiderivative(0.0)) / Z_RAW)  # = omega_c*1 (int S = 1)


def spectrum(w):
    """Normalised truncated double Lorentzian S(omega); zero outside [0, 8]."""
    w = np.asarray(w, dtype=np.float64)
    raw = sum(wt * g / ((w - w0) ** 2 + g * g) for wt, w0, g in _PEAKS) / Z_RAW
    return np.where((w >= 0.0) & (w <= _SUPPORT), raw, 0.0)


def bin_averages(omega_edges_left, domega):
    """Exact bin averages (1/domega) int_bin S dw of the truncated spectrum (atan closed form)."""
    lo = np.clip(np.asarray(omega_edges_left, dtype=np.float64), 0.0, _SUPPORT)
    hi = np.clip(np.asarray(omega_edges_left, dtype=np.float64) + domega, 0.0, _SUPPORT)
    return (_raw_cdf(hi) - _raw_cdf(lo)) / Z_RAW / domega


def correlation_simpson(tau, n_intervals=1_000_000, chunk=8):
    """F(tau_j) = (1/2pi) int_0^8 S(w) exp(-w tau_j) dw, composite Simpson on n_intervals (even)."""
    assert n_intervals % 2 == 0
    tau = np.asarray(tau, dtype=np.float64)
    w = np.linspace(0.0, _SUPPORT, n_intervals + 1)
    h = _SUPPORT / n_intervals
    coef = np.full(n_intervals + 1, 2.0)
    coef[1::2] = 4.0
    coef[0] = coef[-1] = 1.0
    sw = spectrum(w) * coef * (h / 3.0) / TWO_PI
    out = np.empty_like(tau)
    for j0 in range(0, tau.size, chunk):
        t = tau[j0:j0 + chunk]
        out[j0:j0 + chunk] = np.exp(-np.outer(t, w)) @ sw
    return out


def geometric_schedule(t0, t1, n_sweeps):
    """T_s = t0*(t1/t0)^(s/(S-1)), s = 0..S-1; a single sweep gets t0."""
    if n_sweeps == 1:
        return np.array([t0], dtype=np.float64)
    s = np.arange(n_sweeps, dtype=np.float64)
    return t0 * (t1 / t0) ** (s / (n_sweeps - 1))


# --- workload description ----------------------------------------------------------------
@dataclass
class Workload:
    name: str
    n_omega: int
    omega_max: float
    n_tau: int
    dtau: float
    eps: float
    noise_seed: int
    W: int
    n_sweeps: int
    t0: float
    t1: float
    branch_every: int = 0       # 0 = no branching
    resync_every: int = 0       # 0 = never
    t_imprint: float = 0.1      # paper default
    rng_seed: int = 0x5A11      # Philox key of the anneal itself
    # filled by build():
    omega: np.ndarray = field(default=None, repr=False)
    tau: np.ndarray = field(default=None, repr=False)
    F_clean: np.ndarray = field(default=None, repr=False)
    F: np.ndarray = field(default=None, repr=False)
    sigma: np.ndarray = field(default=None, repr=False)
    A: float = 0.0
    B: float = 0.0
    eta: float = 0.0
    schedule: np.ndarray = field(default=None, repr=False)

    @property
    def domega(self):
        return self.omega_max / self.n_omega

    def build(self, simpson_intervals=1_000_000):
        self.omega = np.arange(self.n_omega, dtype=np.float64) * self.domega
        self.tau = np.arange(self.n_tau, dtype=np.float64) * self.dtau
        self.F_clean = correlation_simpson(self.tau, simpson_intervals)
        xi = np.random.Generator(np.random.Philox(self.noise_seed)).standard_normal(self.n_tau)
        self.F = self.F_clean * (1.0 + self.eps * xi)
        self.sigma = self.eps * self.F_clean
        self.A = float(self.F[0]) * TWO_PI / self.domega
        self.B = FIRST_MOMENT / self.domega
        self.eta = 4.0 / self.n_omega
        self.schedule = geometric_schedule(self.t0, self.t1, self.n_sweeps)
        return self

    def attempted_moves(self):
        return self.W * self.n_sweeps * self.n_omega

    def scaled(self, W=None, n_sweeps=None):
        """Same problem with fewer walkers / sweeps (parity-test sized); schedule recomputed."""
        import copy
        w = copy.copy(self)
        if W is not None:
            w.W = W
        if n_sweeps is not None:
            w.n_sweeps = n_sweeps
            w.schedule = geometric_schedule(w.t0, w.t1, n_sweeps)
        return w


_CONFIGS = {
    # BASELINE.json configs[0..4]; T ranges for branching/noise/stress per SURVEY G9.
    "tiny": dict(n_omega=64, omega_max=8.0, n_tau=32, dtau=0.05, eps=1e-4, noise_seed=1,
                 W=64, n_sweeps=2000, t0=1.0, t1=1e-4),
    "small": dict(n_omega=256, omega_max=8.0, n_tau=100, dtau=0.04, eps=1e-4, noise_seed=2,
                  W=4096, n_sweeps=5000, t0=1.0, t1=1e-5),
    "branching": dict(n_omega=512, omega_max=10.0, n_tau=200, dtau=0.025, eps=1e-5, noise_seed=3,
                      W=65536, n_sweeps=10000, t0=1.0, t1=1e-5, branch_every=100),
    "noise": dict(n_omega=1024, omega_max=10.0, n_tau=256, dtau=0.02, eps=1e-4, noise_seed=5,
                  W=16384, n_sweeps=5000, t0=1.0, t1=1e-5, branch_every=100),
    "stress": dict(n_omega=2048, omega_max=12.0, n_tau=512, dtau=0.01, eps=1e-5, noise_seed=8,
                   W=262144, n_sweeps=1000, t0=1.0, t1=1e-5, branch_every=50, resync_every=200),
}
NOISE_SWEEP = ((1e-3, 4), (1e-4, 5), (1e-5, 6), (1e-6, 7))  # (eps, seed), configs[3]


def make(name, simpson_intervals=1_000_000, **overrides):
    """Build one of the five BASELINE.json workloads (optionally overriding fields, e.g. eps/noise_seed)."""
    cfg = dict(_CONFIGS[name])
    cfg.update(overrides)
    return Workload(name=name, **cfg).build(simpson_intervals)


def random_problem(seed, n_omega, n_tau, omega_max=6.0, dtau=0.07, eps=1e-3):
    """Small random-ish problem for property tests: same spectrum, arbitrary grid sizes."""
    w = Workload(name=f"rand{seed}", n_omega=n_omega, omega_max=omega_max, n_tau=n_tau, dtau=dtau,
                 eps=eps, noise_seed=seed, W=4, n_sweeps=4, t0=1.0, t1=0.1)
    return w.build(simpson_intervals=20_000)
