"""CPU oracle of the SAIL hot path — TEST INFRASTRUCTURE (see oracle/sail_oracle.c header).

Thin ctypes wrapper over `sail_oracle.c` (plain C, fp64, -ffp-contract=off).  Only tests/,
`__graft_entry__.smoke()` and bench.py's cpu_baseline / `--impl reference` legs may import this.
It imports nothing from the CUDA package.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "sail_oracle.c")
_LIB = os.path.join(_HERE, "libsail_oracle.so")


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (strict IEEE: no FMA contraction, no fast-math)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = f"{_LIB}.{os.getpid()}.tmp"      # atomic: concurrent processes (gloo tests) never see a partial file
        cmd = ["gcc", "-O2", "-std=c11", "-ffp-contract=off", "-fno-fast-math", "-fopenmp", "-fPIC",
               "-shared", "-o", tmp, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
        os.replace(tmp, _LIB)
    return _LIB


class _Problem(C.Structure):
    _fields_ = [("n_omega", C.c_int32), ("n_tau", C.c_int32),
                ("omega", C.c_void_p), ("K", C.c_void_p), ("F", C.c_void_p), ("sigma", C.c_void_p),
                ("A", C.c_double), ("B", C.c_double), ("eta", C.c_double),
                ("amp_mode", C.c_int32), ("amp_p", C.c_double), ("amp_m", C.c_double),
                ("y_min", C.c_double), ("seed_lo", C.c_uint32), ("seed_hi", C.c_uint32), ("walk_len", C.c_int32), ("walk_uniform", C.c_double)]


TRACE_DTYPE = np.dtype([("p", "<i4"), ("s", "<i4"), ("flags", "<i4"), ("move", "<i4"),
                        ("rho", "<f8"), ("delta_p", "<f8"), ("delta_s", "<f8"), ("dchi2", "<f8"),
                        ("ln_u", "<f8"), ("ap_new", "<f8"), ("as_new", "<f8"), ("l1", "<f8")])

_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.orc_domega.restype = C.c_double
        _lib.orc_chi2.restype = C.c_double
        _lib.orc_amp_factor.restype = C.c_double
        _lib.orc_amp_factor.argtypes = [C.c_double] * 4
        _lib.orc_branch.restype = C.c_int64
        _lib.orc_num_threads.restype = C.c_int
        _lib.orc_branch_zeros.restype = C.c_int64
    return _lib


def _p(arr):
    return arr.ctypes.data_as(C.c_void_p)


def _f64(x):
    return np.ascontiguousarray(x, dtype=np.float64)


def num_threads() -> int:
    return int(lib().orc_num_threads())


def selfcool_temperature(b, chi2_0, chi2_ave, chi2_min, n_boil, n_ramp, T_start=10.0, freeze_rate=1.0):
    """Self-cooling, temperature of block b = 0, 1, ... from the residues
    the population has reached (chi2_ave, chi2_min: measured after block b-1), readings C1-C3 of DESIGN.md:
      block 0            T = T_start * chi2_0          (unit of T = starting residue, T_start = 10, :216)
      boil   (b <= n_boil)        T = chi2_ave         ("we set T close chi2_ave")
      ramp   (next n_ramp blocks) T goes linearly from chi2_ave to chi2_min ("slowly ramped towards chi2_min")
      freeze (afterwards)         T = chi2_min / (1 + freeze_rate * steps), steps = blocks since the ramp ended
                                  ("lowered below the minimal residue ... proportionately to the number of steps")."""
    if b == 0:
        return T_start * chi2_0
    if b <= n_boil:
        return chi2_ave
    if b <= n_boil + n_ramp:
        f = (b - n_boil) / n_ramp
        return chi2_ave + (chi2_min - chi2_ave) * f
    return chi2_min / (1.0 + freeze_rate * (b - n_boil - n_ramp))


def branching_strength_scale(rate, rate_max):
    """Reading B7 of PAPER.md:184 ("reducing the imprinting strength and the branching fraction according to the
    decrease of the acceptance probability"): the factor both are multiplied by is the block's acceptance rate
    relative to the largest block acceptance rate seen so far (which includes this block's).  0 when nothing has been
    accepted yet."""
    return rate / rate_max if rate_max > 0.0 else 0.0


def stencil(a, s):
    """Eq. 27-29 on one spectrum (no renormalisation)."""
    a = _f64(a)
    out = np.empty_like(a)
    lib().orc_stencil(C.c_int(a.size), C.c_double(s), _p(a), _p(out))
    return out


def philox4x32_10(ctr, key):
    c = np.asarray(ctr, dtype=np.uint32)
    k = np.asarray(key, dtype=np.uint32)
    out = np.zeros(4, dtype=np.uint32)
    lib().orc_philox4x32_10(_p(c), _p(k), _p(out))
    return out


def cvec(omega, tau):
    omega, tau = _f64(omega), _f64(tau)
    c = np.empty(tau.size)
    lib().orc_cvec(C.c_int(omega.size), _p(omega), C.c_int(tau.size), _p(tau), _p(c))
    return c


def kernel_table(omega, tau):
    omega, tau = _f64(omega), _f64(tau)
    K = np.empty((omega.size, tau.size))
    lib().orc_kernel_table(C.c_int(omega.size), _p(omega), C.c_int(tau.size), _p(tau), _p(K))
    return K


def forward(K, a):
    K, a = _f64(K), _f64(a)
    M = np.empty(K.shape[1])
    lib().orc_forward(C.c_int(K.shape[0]), C.c_int(K.shape[1]), _p(K), _p(a), _p(M))
    return M


def chi2(M, F, sigma=None):
    M, F = _f64(M), _f64(F)
    sg = _f64(sigma) if sigma is not None else None
    return float(lib().orc_chi2(C.c_int(M.size), _p(M), _p(F), _p(sg) if sg is not None else None))


def init_tilt(omega, A, B):
    omega = _f64(omega)
    a = np.empty(omega.size)
    rc = lib().orc_init_tilt(C.c_int(omega.size), _p(omega), C.c_double(A), C.c_double(B), _p(a))
    if rc != 0:
        raise ValueError("B/A outside the frequency grid")
    return a


def amp_factor(acc_rate, amp_p=1.0, amp_m=2.0, y_min=1e-6):
    return float(lib().orc_amp_factor(acc_rate, amp_p, amp_m, y_min))


class Oracle:
    """State of W walkers + the problem; methods follow include/sail.h call for call."""

    def __init__(self, omega, tau, F, sigma, A, B, eta, seed, amp_mode=1, amp_p=1.0, amp_m=2.0,
                 y_min=1e-6, walk_len=0, walk_uniform=0.0):
        self.omega, self.tau, self.F = _f64(omega), _f64(tau), _f64(F)
        self.sigma = _f64(sigma) if sigma is not None else np.ones_like(self.F)
        self.K = kernel_table(self.omega, self.tau)
        self.n_omega, self.n_tau = self.omega.size, self.tau.size
        self.P = _Problem(self.n_omega, self.n_tau, self.omega.ctypes.data, self.K.ctypes.data,
                          self.F.ctypes.data, self.sigma.ctypes.data, A, B, eta, amp_mode, amp_p,
                          amp_m, y_min, seed & 0xFFFFFFFF, (seed >> 32) & 0xFFFFFFFF, walk_len, walk_uniform)
        self.A, self.B = A, B
        self.sweep = 0
        self.W = 0

    # --- sail_init_walkers -------------------------------------------------------------
    def init_walkers(self, W, spectra=None):
        self.W = W
        if spectra is None:
            self.a = np.tile(init_tilt(self.omega, self.A, self.B), (W, 1))
        else:
            self.a = _f64(spectra).reshape(W, self.n_omega).copy()
        self.M = np.empty((W, self.n_tau))
        self.chi2 = np.empty(W)
        self.y = np.ones(W)
        self.acc = np.zeros(W, dtype=np.int64)
        self.feas = np.zeros(W, dtype=np.int64)
        self.sweep = 0
        self.resync()

    def branch_zeros(self, T):
        """Number of zero multipliers the comb of O8 gives at temperature T (state untouched)."""
        return int(lib().orc_branch_zeros(C.byref(self.P), C.c_int64(self.W), _p(self.chi2), C.c_double(T), C.c_int64(self.sweep)))

    def branch_fraction(self, fraction, t_imprint):
        """f2: find 1/T so that `fraction` of the walkers get multiplier zero (reading B6), then branch at that T.
        Returns (T, n_recipients, mult, donor); T = 0 means no event (degenerate population)."""
        T = C.c_double(0.0)
        ok = lib().orc_branch_fraction_T(C.byref(self.P), C.c_int64(self.W), _p(self.chi2), C.c_double(fraction),
                                         C.c_int64(self.sweep), C.byref(T))
        if not ok:
            return 0.0, 0, None, None
        n_rec, mult, donor = self.branch(T.value, t_imprint)
        return T.value, n_rec, mult, donor

    def resync(self):
        lib().orc_resync(C.byref(self.P), C.c_int64(self.W), _p(self.a), _p(self.M), _p(self.chi2))

    def anneal_selfcool(self, n_blocks, sweeps_per_block, n_boil, n_ramp, t_imprint=0.1, smooth_s=0.0,
                        T_start=10.0, freeze_rate=1.0, T_override=None, branch_fraction=0.0, adapt=False):
        """The paper's block protocol (:218-220) with self-cooling: per block, T from the population's residues, then
        smoothing (if smooth_s > 0; :199), sweeps_per_block sweeps at that T, one branching event at 1/T (or, with
        branch_fraction > 0, at the 1/T that gives that fraction of walkers multiplier zero: the paper's 1/4, :220).  T_override[b]
        replaces the rule (used by the parity tests to drive both sides with the same temperatures).
        Returns (T, chi2_ave, chi2_min) per block."""
        chi2_0 = float(np.mean(self.chi2))
        Ts, aves, mins = [], [], []
        acc_prev, acc_max = int(self.acc.sum()), 0.0
        for b in range(n_blocks):
            ave, mn = float(np.mean(self.chi2)), float(np.min(self.chi2))
            T = selfcool_temperature(b, chi2_0, ave, mn, n_boil, n_ramp, T_start, freeze_rate)
            if T_override is not None:
                T = float(T_override[b])
            Ts.append(T); aves.append(ave); mins.append(mn)
            # reading C3 as amended in round 3 ("Once the transforms are smoothed and renormalized, they
            # undergo Metropolis updates and branching.  The process is then repeated."): smoothing opens the block, so
            # the k sweeps relax what the stencil damaged before the branching weighs the walkers
            if smooth_s > 0.0:
                self.smooth(smooth_s)
            self.anneal(np.full(sweeps_per_block, T))
            scale = 1.0
            if adapt:       # :184, reading B7: strength follows the block's acceptance rate relative to the largest seen
                acc_now = int(self.acc.sum())
                rate = (acc_now - acc_prev) / (float(self.W) * float(sweeps_per_block) * float(self.P.n_omega))
                acc_prev = acc_now
                acc_max = max(acc_max, rate)
                scale = branching_strength_scale(rate, acc_max)
            if branch_fraction > 0.0:
                self.branch_fraction(branch_fraction * scale, t_imprint * scale)
            else:
                self.branch(T, t_imprint * scale)
        return np.array(Ts), np.array(aves), np.array(mins)

    def smooth(self, s):
        """Eq. 27-29 + renormalisation of the second sum rule (reading S2) + resync, all walkers."""
        lib().orc_smooth(C.byref(self.P), C.c_int64(self.W), C.c_double(s), _p(self.a), _p(self.M), _p(self.chi2))

    # --- sail_anneal -------------------------------------------------------------------
    def anneal(self, T_sched, resync_every=0, trace_walkers=None, want_flags=False):
        T = _f64(T_sched)
        n = T.size
        trace = None
        lo = hi = 0
        if trace_walkers is not None:
            lo, hi = trace_walkers
            trace = np.zeros((hi - lo, n, self.n_omega), dtype=TRACE_DTYPE)
        flags = np.zeros((self.W, n, self.n_omega), dtype=np.uint8) if want_flags else None
        lib().orc_anneal(C.byref(self.P), C.c_int64(self.W), _p(self.a), _p(self.M), _p(self.chi2),
                         _p(self.y), _p(T), C.c_int64(self.sweep), C.c_int64(n),
                         C.c_int64(resync_every), _p(self.acc), _p(self.feas),
                         C.c_int64(lo), C.c_int64(hi),
                         _p(trace) if trace is not None else None,
                         _p(flags) if flags is not None else None)
        self.sweep += n
        return trace, flags

    def move(self, walker, sweep, move, T, y=None):
        """One attempted move of one walker (O5); returns the trace record."""
        tr = np.zeros(1, dtype=TRACE_DTYPE)
        yy = float(self.y[walker] if y is None else y)
        c2 = C.c_double(self.chi2[walker])
        lib().orc_move(C.byref(self.P), C.c_int64(walker), C.c_int64(sweep), C.c_int32(move),
                       C.c_double(T), C.c_double(yy), _p(self.a[walker]), _p(self.M[walker]),
                       C.byref(c2), _p(tr))
        self.chi2[walker] = c2.value
        return tr[0]

    def move_raw(self, walker_id, sweep, move, T, a, M, y=1.0):
        """orc_move on caller-supplied arrays (a [n_omega], M [n_tau]); the object's state is not touched."""
        tr = np.zeros(1, dtype=TRACE_DTYPE)
        c2 = C.c_double(0.0)
        lib().orc_move(C.byref(self.P), C.c_int64(walker_id), C.c_int64(sweep), C.c_int32(move),
                       C.c_double(T), C.c_double(y), _p(a), _p(M), C.byref(c2), _p(tr))
        return tr[0]

    # --- sail_branch -------------------------------------------------------------------
    def branch(self, T, t_imprint):
        mult = np.zeros(self.W, dtype=np.int32)
        donor = np.zeros(self.W, dtype=np.int64)
        n_rec = lib().orc_branch(C.byref(self.P), C.c_int64(self.W), _p(self.a), _p(self.M),
                                 _p(self.chi2), C.c_double(T), C.c_double(t_imprint),
                                 C.c_int64(self.sweep), _p(mult), _p(donor))
        return int(n_rec), mult, donor
