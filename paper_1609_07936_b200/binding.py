"""Thin ctypes binding of libsail_b200.so (include/sail.h) — argument marshalling only.

Every numerical step runs in the library's CUDA kernels.  PyTorch is used for device memory (the
workspace and trace buffers are torch tensors) and for the stream.  There is NO fallback: if the
shared library is missing or no CUDA device is visible, calls raise.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libsail_b200.so")

SAIL_OK, SAIL_ERR_ARG, SAIL_ERR_GRID, SAIL_ERR_ALLOC, SAIL_ERR_CUDA, SAIL_ERR_STATE = 0, -1, -2, -3, -4, -5

EXPORTS = ["sail_workspace_bytes", "sail_create", "sail_init_walkers", "sail_anneal", "sail_branch",
           "sail_resync", "sail_get", "sail_get_model", "sail_stats", "sail_set_walkers", "sail_set_sweep",
           "sail_destroy", "sail_last_error", "sail_launch_count", "sail_measure_fp64_peak", "sail_microbench", "sail_smooth", "sail_chi2_stats", "sail_anneal_selfcool", "sail_branch_fraction", "sail_set_walker_offset", "sail_set_chi2",
           "sail_chi2_stats_static"]


class SailError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"sail error {code}: {msg}")
        self.code = code


class sail_config(C.Structure):
    _fields_ = [("device", C.c_int32), ("reserved", C.c_int32), ("stream", C.c_void_p),
                ("workspace", C.c_void_p), ("workspace_bytes", C.c_size_t), ("max_walkers", C.c_int64)]


class sail_anneal_params(C.Structure):
    _fields_ = [("eta", C.c_double), ("amp_mode", C.c_int32), ("reserved0", C.c_int32),
                ("amp_p", C.c_double), ("amp_m", C.c_double), ("y_min", C.c_double),
                ("resync_every", C.c_int64), ("trace_lo", C.c_int64), ("trace_hi", C.c_int64),
                ("trace", C.c_void_p), ("flags", C.c_void_p), ("walk_length", C.c_int32), ("reserved", C.c_int32),
                ("walk_uniform", C.c_double)]


class sail_selfcool_params(C.Structure):
    _fields_ = [("sweeps_per_block", C.c_int32), ("n_boil", C.c_int32), ("n_ramp", C.c_int32),
                ("T_start", C.c_double), ("freeze_rate", C.c_double), ("t_imprint", C.c_double),
                ("smooth_s", C.c_double), ("branch", C.c_int32), ("adapt", C.c_int32),
                ("branch_fraction", C.c_double), ("T_override", C.c_void_p), ("anneal", sail_anneal_params)]


class sail_branch_info(C.Structure):
    _fields_ = [("n_recipients", C.c_int64), ("max_multiplier", C.c_int32), ("reserved", C.c_int32),
                ("chi2_min", C.c_double)]


TRACE_DTYPE = np.dtype([("p", "<i4"), ("s", "<i4"), ("flags", "<i4"), ("move", "<i4"),
                        ("rho", "<f8"), ("delta_p", "<f8"), ("delta_s", "<f8"), ("dchi2", "<f8"),
                        ("thr", "<f8"), ("ap_new", "<f8"), ("as_new", "<f8")])

_lib = None


def lib():
    """Load libsail_b200.so; raises if it has not been built (python -m paper_1609_07936_b200.build)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(f"{LIB_PATH} is missing: build it with `python -m paper_1609_07936_b200.build` "
                               "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        L.sail_workspace_bytes.restype = C.c_size_t
        L.sail_workspace_bytes.argtypes = [C.c_int32, C.c_int32, C.c_int64]
        L.sail_create.argtypes = [C.POINTER(C.c_void_p), C.c_void_p, C.c_int32, C.c_void_p, C.c_int32,
                                  C.c_void_p, C.c_void_p, C.POINTER(sail_config)]
        L.sail_init_walkers.argtypes = [C.c_void_p, C.c_int64, C.c_double, C.c_double, C.c_uint64, C.c_int32, C.c_void_p]
        L.sail_anneal.argtypes = [C.c_void_p, C.c_void_p, C.c_int64, C.POINTER(sail_anneal_params)]
        L.sail_branch.argtypes = [C.c_void_p, C.c_double, C.c_double, C.POINTER(sail_branch_info), C.c_void_p, C.c_void_p]
        L.sail_resync.argtypes = [C.c_void_p]
        L.sail_smooth.argtypes = [C.c_void_p, C.c_double]
        L.sail_branch_fraction.argtypes = [C.c_void_p, C.c_double, C.c_double, C.POINTER(C.c_double),
                                           C.POINTER(sail_branch_info), C.c_void_p, C.c_void_p]
        L.sail_chi2_stats.argtypes = [C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_double)]
        L.sail_chi2_stats_static.argtypes = [C.c_int32, C.c_void_p, C.c_void_p, C.c_int64, C.c_void_p]
        L.sail_anneal_selfcool.argtypes = [C.c_void_p, C.POINTER(sail_selfcool_params), C.c_int64, C.c_void_p,
                                           C.c_void_p, C.c_void_p]
        L.sail_get.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int32]
        L.sail_get_model.argtypes = [C.c_void_p, C.c_void_p, C.c_int32]
        L.sail_stats.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.sail_set_walkers.argtypes = [C.c_void_p, C.c_int64, C.c_int64, C.c_void_p, C.c_void_p]
        L.sail_set_sweep.argtypes = [C.c_void_p, C.c_int64]
        L.sail_set_walker_offset.argtypes = [C.c_void_p, C.c_int64]
        L.sail_set_chi2.argtypes = [C.c_void_p, C.c_int64, C.c_int64, C.c_void_p]
        L.sail_destroy.argtypes = [C.c_void_p]
        L.sail_last_error.restype = C.c_char_p
        L.sail_last_error.argtypes = [C.c_void_p]
        L.sail_launch_count.restype = C.c_int64
        L.sail_launch_count.argtypes = [C.c_void_p]
        L.sail_measure_fp64_peak.argtypes = [C.c_int32, C.c_void_p, C.POINTER(C.c_double)]
        L.sail_microbench.argtypes = [C.c_int32, C.c_void_p, C.POINTER(C.c_double), C.c_int32]
        _lib = L
    return _lib


def _f64(x):
    return np.ascontiguousarray(x, dtype=np.float64)


def _ptr(arr):
    return arr.ctypes.data_as(C.c_void_p) if arr is not None else None


def measure_fp64_peak(device=0):
    """FP64 fused multiply-adds per second (lane-instructions/s) of a register-resident DFMA loop."""
    import torch
    out = C.c_double(0.0)
    rc = lib().sail_measure_fp64_peak(device, C.c_void_p(torch.cuda.current_stream(device).cuda_stream), C.byref(out))
    if rc:
        raise SailError(rc, lib().sail_last_error(None).decode())
    return out.value


MICROBENCH_KEYS = ("dmul_2op_per_clk_sm", "dfma_const_operand_per_clk_sm", "dfma_3op_reuse_per_clk_sm", "dfma_3op_distinct_per_clk_sm",
                   "dmma_m8n8k4_per_clk_sm", "clk_per_sm_2dmma_8dfma", "shfl_per_clk_sm",
                   "lds128_uniform_per_clk_sm", "lds64_lane_per_clk_sm", "dfma_latency_clk", "shfl_latency_clk",
                   "dmma_latency_clk", "dfma_3op_reuse_per_clk_sm_1warp_per_subpartition", "tau_loop_credited_per_clk_sm",
                   "warp_sum_dmma_latency_clk", "warp_sum_shfl_latency_clk")


def microbench(device=0):
    """Issue rates / latencies behind the sweep-kernel design (include/sail.h: sail_microbench)."""
    import torch
    out = (C.c_double * len(MICROBENCH_KEYS))()
    rc = lib().sail_microbench(device, C.c_void_p(torch.cuda.current_stream(device).cuda_stream), out, len(MICROBENCH_KEYS))
    if rc:
        raise SailError(rc, lib().sail_last_error(None).decode())
    return {k: float(v) for k, v in zip(MICROBENCH_KEYS, out)}


STATS_STATIC_MAX_W = 1 << 24     # include/sail.h: SAIL_STATS_STATIC_MAX_W


def chi2_stats_static(chi2_t, out_t, n=None):
    """(min, mean) of the residues in the CUDA float64 tensor `chi2_t` (first `n` entries; default all) into the
    CUDA float64 tensor `out_t` (2 entries), enqueued on torch's current stream of that device, without a handle and
    without any device allocation: for a thread that watches an anneal from a copy of the residues and can neither
    use the handle (one thread at a time) nor afford cudaMalloc's device-wide wait.  The scratch is one fixed 4 KB
    array per GPU shared by all calls: keep the calls of a device on one stream (include/sail.h:
    sail_chi2_stats_static).  Nothing is copied or synchronised here; read `out_t` when you need the numbers."""
    import torch
    if not (chi2_t.is_cuda and out_t.is_cuda and chi2_t.dtype == torch.float64 and out_t.dtype == torch.float64
            and chi2_t.is_contiguous() and out_t.is_contiguous() and out_t.numel() >= 2
            and chi2_t.device == out_t.device):
        raise ValueError("chi2_t and out_t must be contiguous float64 CUDA tensors on one device, out_t with >= 2 entries")
    n = chi2_t.numel() if n is None else int(n)
    if n > chi2_t.numel():
        raise ValueError("n exceeds the tensor")
    dev = chi2_t.device.index
    rc = lib().sail_chi2_stats_static(dev, C.c_void_p(torch.cuda.current_stream(dev).cuda_stream),
                                      C.c_void_p(chi2_t.data_ptr()), n, C.c_void_p(out_t.data_ptr()))
    if rc:
        raise SailError(rc, lib().sail_last_error(None).decode())


class Sail:
    """One inverse problem + its walker population on one GPU (handle of include/sail.h)."""

    def __init__(self, omega, tau, F, sigma=None, max_walkers=1, device=0, torch_workspace=True):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("sail-b200 needs a CUDA device; there is no CPU fallback")
        L = lib()
        self._L = L
        self.device = device
        omega, tau, F = _f64(omega), _f64(tau), _f64(F)
        sg = _f64(sigma) if sigma is not None else None
        self.n_omega, self.n_tau = omega.size, tau.size
        self.max_walkers = int(max_walkers)
        cfg = sail_config()
        cfg.device = device
        cfg.stream = torch.cuda.current_stream(device).cuda_stream
        cfg.max_walkers = self.max_walkers
        self._ws = None
        if torch_workspace:
            nbytes = L.sail_workspace_bytes(self.n_omega, self.n_tau, self.max_walkers)
            self._ws = torch.empty(nbytes + 256, dtype=torch.uint8, device=f"cuda:{device}")
            base = (self._ws.data_ptr() + 255) & ~255
            cfg.workspace = base
            cfg.workspace_bytes = nbytes
        h = C.c_void_p()
        rc = L.sail_create(C.byref(h), _ptr(omega), self.n_omega, _ptr(tau), self.n_tau, _ptr(F), _ptr(sg), C.byref(cfg))
        if rc:
            raise SailError(rc, L.sail_last_error(None).decode())
        self._h = h
        self.W = 0

    # ------------------------------------------------------------------------------------------
    def _check(self, rc):
        if rc:
            raise SailError(rc, self._L.sail_last_error(self._h).decode())

    def init_walkers(self, W, A, B, seed, spectra=None):
        sp = _f64(spectra) if spectra is not None else None
        if sp is not None and sp.size != W * self.n_omega:
            raise ValueError("spectra must be [W][n_omega]")
        self._check(self._L.sail_init_walkers(self._h, W, A, B, C.c_uint64(seed), 0 if sp is None else 1, _ptr(sp)))
        self.W = W

    def anneal(self, T_schedule, eta, amp_mode=1, amp_p=1.0, amp_m=2.0, y_min=1e-6, resync_every=0,
               trace_walkers=None, want_flags=False, walk_length=0, walk_uniform=0.0):
        """Run len(T_schedule) sweeps.  Returns (trace, flags) numpy arrays when requested, else (None, None)."""
        import torch
        T = _f64(T_schedule)
        p = sail_anneal_params()
        p.eta, p.amp_mode = eta, amp_mode
        p.amp_p, p.amp_m, p.y_min, p.resync_every = amp_p, amp_m, y_min, resync_every
        p.walk_length, p.walk_uniform = walk_length, walk_uniform
        trace_t = flags_t = None
        if trace_walkers is not None:
            lo, hi = trace_walkers
            p.trace_lo, p.trace_hi = lo, hi
            nbytes = (hi - lo) * T.size * self.n_omega * TRACE_DTYPE.itemsize
            trace_t = torch.zeros(nbytes, dtype=torch.uint8, device=f"cuda:{self.device}")
            p.trace = trace_t.data_ptr()
        if want_flags:
            flags_t = torch.zeros(self.W * T.size * self.n_omega, dtype=torch.uint8, device=f"cuda:{self.device}")
            p.flags = flags_t.data_ptr()
        self._check(self._L.sail_anneal(self._h, _ptr(T), T.size, C.byref(p)))
        trace = flags = None
        if trace_t is not None:
            lo, hi = trace_walkers
            trace = trace_t.cpu().numpy().view(TRACE_DTYPE).reshape(hi - lo, T.size, self.n_omega)
        if flags_t is not None:
            flags = flags_t.cpu().numpy().reshape(self.W, T.size, self.n_omega)
        return trace, flags

    def chi2_stats(self):
        """(min, mean) of chi^2 over the population (include/sail.h: sail_chi2_stats)."""
        mn, mean = C.c_double(), C.c_double()
        self._check(self._L.sail_chi2_stats(self._h, C.byref(mn), C.byref(mean)))
        return mn.value, mean.value

    def anneal_selfcool(self, n_blocks, sweeps_per_block, n_boil, n_ramp, eta, t_imprint=0.1, smooth_s=0.0, T_start=10.0,
                        freeze_rate=1.0, branch=True, branch_fraction=0.0, adapt=False, T_override=None, amp_mode=1, amp_p=1.0, amp_m=2.0, y_min=1e-6,
                        resync_every=0, walk_length=0, walk_uniform=0.0):
        """The paper's block protocol with self-cooling (include/sail.h: sail_anneal_selfcool).
        Returns (T, chi2_ave, chi2_min), one entry per block.  resync_every > 0 recomputes the residues from the spectra
        after every such sweep (keeps the running chi2_min the rule feeds on from drifting below zero near an exact fit);
        walk_length / walk_uniform select the index walk of section 2.3 as in anneal()."""
        p = sail_selfcool_params()
        p.sweeps_per_block, p.n_boil, p.n_ramp = sweeps_per_block, n_boil, n_ramp
        p.T_start, p.freeze_rate, p.t_imprint, p.smooth_s, p.branch = T_start, freeze_rate, t_imprint, smooth_s, int(branch)
        p.branch_fraction = branch_fraction
        p.adapt = int(adapt)
        ov = _f64(T_override) if T_override is not None else None
        p.T_override = ov.ctypes.data if ov is not None else None
        p.anneal.eta, p.anneal.amp_mode = eta, amp_mode
        p.anneal.amp_p, p.anneal.amp_m, p.anneal.y_min = amp_p, amp_m, y_min
        p.anneal.resync_every, p.anneal.walk_length, p.anneal.walk_uniform = resync_every, walk_length, walk_uniform
        T, ave, mn = np.zeros(n_blocks), np.zeros(n_blocks), np.zeros(n_blocks)
        self._check(self._L.sail_anneal_selfcool(self._h, C.byref(p), n_blocks, _ptr(T), _ptr(ave), _ptr(mn)))
        return T, ave, mn

    def branch(self, T, t_imprint, want_maps=False):
        info = sail_branch_info()
        mult = np.empty(self.W, dtype=np.int32) if want_maps else None
        donor = np.empty(self.W, dtype=np.int64) if want_maps else None
        self._check(self._L.sail_branch(self._h, T, t_imprint, C.byref(info), _ptr(mult), _ptr(donor)))
        return info, mult, donor

    def branch_fraction(self, fraction, t_imprint, want_maps=False):
        """f2: branch so that `fraction` of the walkers get multiplier zero.  Returns (T_found, info, mult, donor)."""
        info = sail_branch_info()
        T = C.c_double(0.0)
        mult = np.empty(self.W, dtype=np.int32) if want_maps else None
        donor = np.empty(self.W, dtype=np.int64) if want_maps else None
        self._check(self._L.sail_branch_fraction(self._h, C.c_double(fraction), C.c_double(t_imprint), C.byref(T),
                                                 C.byref(info), _ptr(mult), _ptr(donor)))
        return T.value, info, mult, donor

    def branch_async(self, T, t_imprint):
        self._check(self._L.sail_branch(self._h, T, t_imprint, None, None, None))

    def resync(self):
        self._check(self._L.sail_resync(self._h))

    def smooth(self, s):
        """Eq. 27-29 + renormalisation of the second sum rule + resync (include/sail.h: sail_smooth)."""
        self._check(self._L.sail_smooth(self._h, C.c_double(s)))

    def get(self, spectra=True, chi2=True):
        sp = np.empty((self.W, self.n_omega)) if spectra else None
        c2 = np.empty(self.W) if chi2 else None
        self._check(self._L.sail_get(self._h, _ptr(sp), _ptr(c2), 0))
        return sp, c2

    def get_into(self, spectra_host, chi2_host):
        """Copy into caller-provided (e.g. pinned) host arrays."""
        self._check(self._L.sail_get(self._h, _ptr(spectra_host), _ptr(chi2_host), 0))

    def get_device(self, spectra_t=None, chi2_t=None):
        """Stream-ordered copy into torch CUDA tensors (float64)."""
        self._check(self._L.sail_get(self._h, spectra_t.data_ptr() if spectra_t is not None else None,
                                     chi2_t.data_ptr() if chi2_t is not None else None, 1))

    def get_model(self):
        M = np.empty((self.W, self.n_tau))
        self._check(self._L.sail_get_model(self._h, _ptr(M), 0))
        return M

    def stats(self):
        acc = np.empty(self.W, dtype=np.int64)
        ev = np.empty(self.W, dtype=np.int64)
        y = np.empty(self.W)
        self._check(self._L.sail_stats(self._h, _ptr(acc), _ptr(ev), _ptr(y)))
        return acc, ev, y

    def set_walkers(self, w0, spectra, y=None):
        sp = _f64(spectra).reshape(-1, self.n_omega)
        yy = _f64(y) if y is not None else None
        self._check(self._L.sail_set_walkers(self._h, w0, sp.shape[0], _ptr(sp), _ptr(yy)))

    def set_chi2(self, chi2, w0=0):
        """Overwrite the running residues of walkers [w0, w0 + len(chi2))."""
        c2 = _f64(chi2)
        self._check(self._L.sail_set_chi2(self._h, w0, c2.size, _ptr(c2)))

    def set_walker_offset(self, first_walker):
        """Global index of walker 0: sharded populations draw the single-handle random streams."""
        self._check(self._L.sail_set_walker_offset(self._h, first_walker))

    def set_sweep(self, sweep):
        self._check(self._L.sail_set_sweep(self._h, sweep))

    def launch_count(self):
        return int(self._L.sail_launch_count(self._h))

    def close(self):
        if getattr(self, "_h", None):
            self._L.sail_destroy(self._h)
            self._h = None
        self._ws = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
