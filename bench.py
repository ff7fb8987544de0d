#!/usr/bin/env python
"""bench.py — SAIL hot path on B200: attempted walker-moves/s, anneals/s and the roofline fraction.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload stress]

Headline workload: BASELINE.json configs[4] "Throughput stress" (the largest single-GPU configuration; `metric` names
no configuration).  A "step" is ONE PROTOCOL BLOCK of the workload: `branch_every` sweeps of the temperature schedule
(proposal, positivity, Delta chi^2 over all tau, Metropolis, Eq. 30 — one persistent sweep-kernel launch per piece between
resyncs), the full-residual resync where the absolute sweep counter crosses `resync_every`, and the imprinted-branching
event that ends the block; the last block of an anneal adds the final sail_get.  Stress: 20 blocks of 50 sweeps ARE one
whole anneal, so the default K = 20 times exactly one anneal.  (Workloads without branching: a step is the whole anneal.)
The W warm-up steps run the first blocks of the schedule; then the walkers are re-initialised (untimed) and the K timed
steps start at block 0 (again re-initialised, outside the per-step CUDA events, whenever the block index wraps).
`value` is measured with inputs resident in HBM; `e2e` runs the same K steps through the C ABI with HOST buffers
(problem arrays and schedule slices H2D, chi^2 of all walkers D2H after every block, spectra D2H at the end of the
anneal, create / init / destroy inside the timed region).  `configs` holds one whole anneal of each of the five
BASELINE.json configurations.

`--impl reference` times the CPU oracle (oracle/, as it stands) on the host cores on a bounded sample of the same
workload (this tier has no reference implementation to install).
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_1609_07936_b200 import distributed as sdist  # noqa: E402
from paper_1609_07936_b200 import workloads as wl  # noqa: E402

METRIC = "attempted_walker_moves_per_s"
UNIT = "moves/s"
FP64_LANES_PER_SM = 64          # FP64 lanes per SM per clock (4 sub-partitions x 16), see DESIGN.md §6.1
DFMA_PER_TAU_POINT = 5          # algorithmic FP64-pipe instructions per tau-point per evaluated move
NAMES = ["tiny", "small", "branching", "noise", "stress"]

# dram__bytes_read.sum + dram__bytes_write.sum of ONE sweep-kernel launch, from the committed `ncu --set full` captures
# profiles/r02_sweep_{stress,noise,branching,small,tiny}_full_metrics.txt (2-sweep launches).  A warp runs ALL sweeps of a launch on a
# walker while that walker's spectrum and model are resident on chip, so the DRAM traffic of a launch is the walker state
# once in and once out (algorithmic: 16 W (N_omega + N_tau) bytes) whatever the number of sweeps; states that fit the
# 126 MB L2 (small, noise) partly stay there between launches.
SWEEP_DRAM_BYTES_PER_LAUNCH = {"stress": 11.094e9, "noise": 0.2822e9, "branching": 0.6969e9, "small": 11.9e6, "tiny": 92.4e3}


# Whole-anneal sweep-kernel fractions of the NOMINAL FP64 rate in the driver-run lines of the earlier rounds
# (profiles/r01_all_configs.md, profiles/r02_bench_stress.json.txt `configs`), so that a change of the headline workload
# is not read as kernel progress: the headline was Small in round 1 and is Stress since round 2.  This round's figures
# are `configs[*].roofline_frac` of the same line (also of the nominal rate).
HISTORY = {"headline_workload": {"r01": "small", "r02": "stress", "r03": "stress"},
           "sweep_kernel_frac_of_nominal": {"r01": {"tiny": 0.002, "small": 0.177, "branching": 0.280, "noise": 0.305, "stress": 0.395},
                                            "r02": {"tiny": 0.002, "small": 0.173, "branching": 0.278, "noise": 0.305, "stress": 0.398}},
           "note": "r01 -> r02 changed no configuration by more than 0.004: the round-2 headline gain (0.176 -> 0.398) is the workload switch"}


def build_defines():
    """The -D flags the library on disk was built with (paper_1609_07936_b200/build/defines.txt); [] = the product library."""
    try:
        return open(os.path.join(ROOT, "paper_1609_07936_b200", "build", "defines.txt")).read().split()
    except OSError:
        return None


# ------------------------------------------------------------------------------------------------
class ClockSampler:
    """Samples nvidia-smi clocks / throttle reasons during the timed region."""

    FIELDS = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
              "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
              "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.proc, self.lines = index, None, []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.FIELDS}",
                                          "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, reasons, power = [], [], set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for l in self.lines:
            f = [x.strip() for x in l.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1])); power.append(float(f[2]))
            except ValueError:
                continue
            for n, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(power) if power else None, "samples": len(sm), "reasons": sorted(reasons)}


def measured_peaks():
    try:
        return json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        return {}


def host_cores():
    try:
        return len(os.sched_getaffinity(0))
    except Exception:
        return os.cpu_count() or 1


def workload_string(w):
    s = (f"{w.name} (BASELINE.json configs[{NAMES.index(w.name)}]): N_omega={w.n_omega}, N_tau={w.n_tau}, W={w.W}, "
         f"sweeps={w.n_sweeps}, T {w.t0}->{w.t1} geometric, eps={w.eps}")
    if w.branch_every:
        s += f", imprinted branching (t={w.t_imprint}) every {w.branch_every} sweeps"
    if w.resync_every:
        s += f", resync every {w.resync_every} sweeps"
    return s


def anneal_params(w):
    return dict(eta=w.eta, amp_mode=1, amp_p=1.0, amp_m=2.0, y_min=1e-6, resync_every=w.resync_every)


def block_layout(w):
    bs = w.branch_every if w.branch_every else w.n_sweeps
    return bs, (w.n_sweeps + bs - 1) // bs


# ------------------------------------------------------------------------------------------------
def run_block(s, w, b, torch, dev_out=None, host_out=None):
    """Block b of the workload's protocol on an initialised handle.  Returns the CUDA events around the sweep kernels.
    dev_out = (spectra_t, chi2_t): device-side sail_get after the last block; host_out = (spectra_h, chi2_h): chi^2 to
    the host after every block, spectra after the last one."""
    bs, nb = block_layout(w)
    lo, hi = b * bs, min((b + 1) * bs, w.n_sweeps)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    s.anneal(w.schedule[lo:hi], **anneal_params(w))
    e1.record()
    if w.branch_every and hi % w.branch_every == 0:
        s.branch_async(float(w.schedule[hi - 1]), w.t_imprint)
    last = b == nb - 1
    if host_out is not None:
        s.get_into(host_out[0] if last else None, host_out[1])
    elif last and dev_out is not None:
        s.get_device(*dev_out)
    return e0, e1


def l2_is_flushed(w):
    """Small walker states would sit in the 126 MB L2 between steps: they are flushed (256 MiB write) between steps."""
    return 8 * w.W * (w.n_omega + w.n_tau) < 512 * 1024 * 1024


def config_dict(w, world):
    """The `config` object of the JSON line: one definition for our arm and for the reference arm (--impl reference),
    so that both name the same workload and the same step."""
    bs, nb = block_layout(w)
    state_bytes = 8 * w.W * (w.n_omega + w.n_tau)
    return {"workload": workload_string(w),
            "step": (f"one protocol block: {bs} sweeps (+ resync / imprinted branching as configured); {nb} blocks = one whole anneal; "
                     "walkers re-initialised untimed when the block index wraps") if nb > 1 else
                    "one whole anneal (all sweeps + final sail_get), walkers re-initialised untimed",
            "parallelism": f"{world} independent replica(s), one per GPU",
            "l2": "flushed between steps (256 MiB write)" if l2_is_flushed(w) else
                  f"not flushed: the walker state a step streams ({state_bytes / 2**30:.1f} GiB) is larger than L2 (126 MB)",
            "attempted_moves_per_step": w.W * bs * w.n_omega, "blocks_per_anneal": nb}


def cpu_oracle_sample(w, target_s=12.0, seed=0x5A11, whole=False):
    """Oracle (as it stands) on the host cores.  whole = False: a bounded sample (a subset of walkers over the first
    sweeps of the schedule); whole = True: the whole anneal of the workload (Tiny / Small only).
    Returns (moves/s, threads, description)."""
    os.environ.setdefault("OMP_NUM_THREADS", str(host_cores()))
    import oracle
    cores = min(oracle.num_threads(), host_cores())
    o = oracle.Oracle(w.omega, w.tau, w.F, w.sigma, w.A, w.B, w.eta, seed)
    if whole:
        o.init_walkers(w.W)
        t0 = time.perf_counter()
        o.anneal(w.schedule, resync_every=w.resync_every)
        dt = time.perf_counter() - t0
        return w.attempted_moves() / dt, cores, f"whole anneal of '{w.name}' ({w.attempted_moves():.3g} moves, {dt:.1f} s)"
    Ws = max(cores * 8, 64)
    o.init_walkers(Ws)
    probe = 4
    t0 = time.perf_counter()
    o.anneal(w.schedule[:probe], resync_every=w.resync_every)
    dt = time.perf_counter() - t0
    n_sw = int(max(probe, min(w.n_sweeps - probe, target_s / max(dt / probe, 1e-9))))
    t0 = time.perf_counter()
    o.anneal(w.schedule[probe:probe + n_sw], resync_every=w.resync_every)
    dt = time.perf_counter() - t0
    moves = Ws * n_sw * w.n_omega
    return moves / dt, cores, f"{Ws} walkers x sweeps {probe}..{probe + n_sw} of '{w.name}' ({moves:.3g} moves, {dt:.1f} s)"


# ------------------------------------------------------------------------------------------------
def main_reference(args):
    rank, _, world = sdist.env_world()
    if rank != 0:
        return 0
    w = wl.make(args.workload)
    bs, nb = block_layout(w)
    if args.cpu_whole:
        # the oracle on the WHOLE anneal of the workload, once (BASELINE.md asks for it on Tiny and Small; Small takes minutes)
        v, cores, sample = cpu_oracle_sample(w, whole=True)
        print(json.dumps({"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": 1, "warmup": 0,
                          "ms_per_step": 1e3 * w.attempted_moves() / v, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                          "dtype": "f64", "data": "synthetic", "config": {"workload": workload_string(w), "step": "one whole anneal on the CPU oracle"},
                          "cpu_baseline": {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
                          "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}, "gpu_launches": 0}))
        return 0
    vals = []
    for _ in range(args.warmup):
        cpu_oracle_sample(w, target_s=1.0)
    t_per = max(2.0, min(20.0, 90.0 / max(args.steps, 1)))
    for _ in range(args.steps):
        v, cores, sample = cpu_oracle_sample(w, target_s=t_per)
        vals.append(v)
    value = float(np.mean(vals))
    step_moves = w.W * bs * w.n_omega
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * step_moves / value,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": config_dict(w, max(args.gpus, 1)),
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle",
                             "sample": sample + f"; one such bounded sample per step, {args.steps} steps, value = their mean; ms_per_step = the "
                                                "time of one step of `config` (a protocol block) at that rate, extrapolated, not run"},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))
    return 0


def main_selfcool(args):
    """Supplementary: the paper's own protocol (self-cooling, blocks of 100 sweeps, smoothing, a quarter of the walkers
    branched with t = 0.1, strength following the acceptance rate) on the chosen workload; prints the trajectory."""
    import torch
    from paper_1609_07936_b200 import build
    build.build(defines=None if args.diag_defines else ())
    from paper_1609_07936_b200.binding import Sail
    w = wl.make(args.workload)
    s = Sail(w.omega, w.tau, w.F, w.sigma, max_walkers=w.W)
    s.init_walkers(w.W, w.A, w.B, w.rng_seed)
    nb, k = args.selfcool, 100
    kw = dict(n_boil=max(1, nb // 10), n_ramp=max(1, nb // 5), eta=w.eta, t_imprint=0.1, smooth_s=0.01, branch_fraction=0.25,
              adapt=True, freeze_rate=0.5)
    torch.cuda.synchronize()
    l0 = s.launch_count()
    t0 = time.perf_counter()
    T, ave, mn = s.anneal_selfcool(nb, k, **kw)
    torch.cuda.synchronize()
    dt = time.perf_counter() - t0
    mn_end, ave_end = s.chi2_stats()
    acc, ev, _ = s.stats()
    print(json.dumps({"protocol": "self-cooling (sail_anneal_selfcool)", "workload": w.name, "blocks": nb, "sweeps_per_block": k,
                      "parameters": {a: b for a, b in kw.items() if a != "eta"}, "seconds": dt, "kernel_launches": s.launch_count() - l0,
                      "attempted_moves_per_s": w.W * nb * k * w.n_omega / dt, "accepted_fraction": float(acc.sum()) / (w.W * nb * k * w.n_omega),
                      "T": [float(x) for x in T], "chi2_ave": [float(x) for x in ave], "chi2_min": [float(x) for x in mn],
                      "chi2_ave_end": ave_end, "chi2_min_end": mn_end, "n_tau": w.n_tau}))
    s.close()
    return 0


def spawn_ranks(args):
    """`python bench.py --gpus N` without a torchrun environment: start N ranks (one per GPU) of this same command."""
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(29500 + os.getpid() % 400), os.path.abspath(__file__)] + sys.argv[1:]
    return subprocess.call(cmd)


def whole_anneal(torch, Sail, w, dev_index, peak, seed):
    """One whole anneal (all blocks) of workload w, device-resident; returns the per-config entry of `configs`."""
    dev = f"cuda:{dev_index}"
    spectra_t = torch.empty((w.W, w.n_omega), dtype=torch.float64, device=dev)
    chi2_t = torch.empty(w.W, dtype=torch.float64, device=dev)
    s = Sail(w.omega, w.tau, w.F, w.sigma, max_walkers=w.W, device=dev_index)
    bs, nb = block_layout(w)
    s.init_walkers(w.W, w.A, w.B, seed)
    if nb > 1:
        run_block(s, w, 0, torch)                         # warm-up: the first block
    else:
        s.anneal(w.schedule[:max(1, min(50, w.n_sweeps // 10))], **anneal_params(w))
    s.init_walkers(w.W, w.A, w.B, seed)
    torch.cuda.synchronize()
    sampler = ClockSampler(dev_index)
    sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    l0 = s.launch_count()
    e0.record()
    kev = [run_block(s, w, b, torch, dev_out=(spectra_t, chi2_t)) for b in range(nb)]
    e1.record()
    torch.cuda.synchronize()
    clocks = sampler.stop()
    t = e0.elapsed_time(e1) * 1e-3
    tk = sum(a.elapsed_time(b) for a, b in kev) * 1e-3
    acc, ev, _ = s.stats()
    entry = {"workload": workload_string(w), "seconds_per_anneal": t, "anneals_per_s": 1.0 / t,
             "value": w.attempted_moves() / t, "unit": UNIT, "evaluated_fraction": float(ev.sum()) / w.attempted_moves(),
             "accepted_fraction": float(acc.sum()) / w.attempted_moves(), "sweep_kernel_seconds": tk,
             "roofline_frac": DFMA_PER_TAU_POINT * w.n_tau * float(ev.sum()) / tk / peak,
             "gpu_launches": s.launch_count() - l0, "chi2_final_median": float(torch.median(chi2_t).item()),
             "clocks": clocks}
    s.close()
    return entry


def main_ours(args):
    import torch
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (no CPU fallback); use --impl reference for the oracle")
    from paper_1609_07936_b200 import build
    build.build(defines=None if args.diag_defines else ())
    from paper_1609_07936_b200.binding import Sail, measure_fp64_peak

    rank, local_rank, world = sdist.init("nccl")
    if local_rank >= torch.cuda.device_count():
        raise SystemExit(f"bench.py: rank {rank} needs cuda:{local_rank} but this node has {torch.cuda.device_count()} GPU(s)")
    torch.cuda.set_device(local_rank)
    dev = f"cuda:{local_rank}"
    w = wl.make(args.workload)
    if args.sweeps:
        w = w.scaled(n_sweeps=args.sweeps)
    bs, nb = block_layout(w)
    seed = sdist.rank_seed(w.rng_seed, rank)          # every rank anneals an independent replica (weak scaling)
    peaks = measured_peaks()
    state_bytes = 8 * w.W * (w.n_omega + w.n_tau)
    l2_flush = l2_is_flushed(w)

    spectra_t = torch.empty((w.W, w.n_omega), dtype=torch.float64, device=dev)
    chi2_t = torch.empty(w.W, dtype=torch.float64, device=dev)
    flush = torch.empty(256 * 1024 * 1024 // 4, dtype=torch.float32, device=dev) if l2_flush else None
    s = Sail(w.omega, w.tau, w.F, w.sigma, max_walkers=w.W, device=local_rank)

    def one_step(i):
        b = i % nb
        if b == 0:
            s.init_walkers(w.W, w.A, w.B, seed)        # untimed set-up of an anneal (A1)
        if flush is not None:
            flush.zero_()                               # L2 flush between timed iterations
        torch.cuda.synchronize()
        l0 = s.launch_count()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        k0, k1 = run_block(s, w, b, torch, dev_out=(spectra_t, chi2_t))
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) * 1e-3, k0.elapsed_time(k1) * 1e-3, s.launch_count() - l0

    for i in range(args.warmup):
        one_step(i)
    sampler = ClockSampler(local_rank)
    sdist.barrier(dev)
    torch.cuda.synchronize()
    sampler.start()
    step_s, kern_s, launches = [], [], 0
    evaluated = accepted = 0.0
    for i in range(args.steps):
        t, k, lc = one_step(i)
        step_s.append(t); kern_s.append(k); launches += lc
        if (i + 1) % nb == 0 or i == args.steps - 1:    # sail_stats counts since the last init: read at the end of an anneal
            acc, ev, _ = s.stats()
            evaluated += float(ev.sum())
            accepted += float(acc.sum())
    torch.cuda.synchronize()
    sdist.barrier(dev)
    clocks = sampler.stop()
    chi2_final = chi2_t.cpu().numpy()
    if args.profile_sweeps:
        # the target of the ncu captures under profiles/: walkers re-initialised, sweeps [0, S) of the schedule in one
        # launch (no branching), then ONE short launch of N sweeps at sweep S = --profile-at (default: mid-anneal).
        # ncu: `-k regex:sweep_kernel -s <launches before> -c 1`; a whole block is seconds long and far too slow to replay
        at = args.profile_at if args.profile_at >= 0 else w.n_sweeps // 2
        at = max(0, min(at, w.n_sweeps - args.profile_sweeps))
        s.init_walkers(w.W, w.A, w.B, seed)
        if at:
            s.anneal(w.schedule[:at], **dict(anneal_params(w), resync_every=0))
        torch.cuda.synchronize()
        s.anneal(w.schedule[at:at + args.profile_sweeps], **dict(anneal_params(w), resync_every=0))
        torch.cuda.synchronize()
    step_moves = w.W * bs * w.n_omega
    total_s, total_moves = sdist.reduce_timing(float(np.sum(step_s)), float(step_moves * args.steps), dev)
    value = total_moves / total_s
    ms_per_step = 1e3 * total_s / args.steps

    # ---- end to end through the C ABI with host buffers: the same K steps, on every rank ------------------
    e2e = None
    if args.e2e:
        host_sp = torch.empty((w.W, w.n_omega), dtype=torch.float64).pin_memory().numpy()
        host_c2 = torch.empty(w.W, dtype=torch.float64).pin_memory().numpy()
        n_e2e = args.steps if args.e2e < 0 else min(args.steps, args.e2e)
        torch.cuda.synchronize()
        sdist.barrier(dev)
        s2 = None
        t0 = time.perf_counter()
        for i in range(n_e2e):
            b = i % nb
            if b == 0:
                if s2 is not None:
                    s2.close()
                s2 = Sail(w.omega, w.tau, w.F, w.sigma, max_walkers=w.W, device=local_rank)     # H2D of the problem
                s2.init_walkers(w.W, w.A, w.B, seed)
            run_block(s2, w, b, torch, host_out=(host_sp, host_c2))    # schedule slice H2D, chi^2 (and spectra) D2H
        torch.cuda.synchronize()
        s2.close()
        dt = time.perf_counter() - t0
        # every rank runs its replica through host buffers: max time over ranks, units of all ranks (whole-job rate)
        dt_max, units_all = sdist.reduce_timing(dt, float(step_moves * n_e2e), dev)
        if n_e2e == args.steps and args.steps % nb == 0:
            assert np.array_equal(host_c2, chi2_final), "e2e run is not bit-identical to the device-resident run"
        n_anneals = max(1, (n_e2e + nb - 1) // nb)
        h2d = 8 * bs + 8 * (w.n_omega + 3 * w.n_tau) * n_anneals / n_e2e
        d2h = 8 * w.W + 8 * w.W * w.n_omega * (n_e2e // nb) / n_e2e
        e2e = {"value": units_all / dt_max, "unit": UNIT, "h2d_bytes_per_step": world * h2d, "d2h_bytes_per_step": world * d2h,
               "steps": n_e2e, "ms_per_step": 1e3 * dt_max / n_e2e,
               "includes": "sail_create + sail_init_walkers at the first block of an anneal, per block: schedule slice H2D, sweeps, resync, "
                           "branching, chi^2 of all walkers to pinned host memory; spectra to the host after the last block; sail_destroy"}


    line = None
    if rank == 0:
        # ---- roofline of the dominant kernel (the sweep kernel): FP64 ALU bound ----------------------
        sm_max = peaks.get("sm_max_mhz") or clocks.get("sm_max_mhz") or 1965.0
        num_sms = torch.cuda.get_device_properties(local_rank).multi_processor_count
        peak_nominal = num_sms * FP64_LANES_PER_SM * sm_max * 1e6
        dfma_measured = measure_fp64_peak(local_rank)
        kern_total = float(np.sum(kern_s))
        achieved = DFMA_PER_TAU_POINT * w.n_tau * evaluated / kern_total
        attempted = float(step_moves * args.steps)
        # the denominator is the DFMA rate MEASURED in this run (register-resident two-operand DFMA chains,
        # sail_measure_fp64_peak); the nominal rate (unit count x clock) is kept beside it
        roofline = {"bound": "alu", "kernel": "sail::sweep_kernel", "achieved": achieved / 1e12, "peak": dfma_measured / 1e12,
                    "unit": "T FP64 lane-instr/s", "frac": achieved / dfma_measured,
                    "traffic": SWEEP_DRAM_BYTES_PER_LAUNCH.get(w.name),
                    "traffic_source": (f"not from this run: dram__bytes_read.sum + dram__bytes_write.sum of one sweep-kernel launch in the committed "
                                       f"`ncu --set full` capture profiles/r02_sweep_{w.name}_full_metrics.txt (a 2-sweep launch; the traffic of a launch "
                                       "is the walker state once in and once out whatever its number of sweeps)"),
                    "peak_source": "measured in this run: sail_measure_fp64_peak, register-resident DFMA chains (FP64 is not in MEASURED_PEAKS.json)",
                    "peak_nominal": peak_nominal / 1e12, "frac_of_nominal": achieved / peak_nominal,
                    "peak_nominal_source": f"derived: {num_sms} SMs x {FP64_LANES_PER_SM} FP64 lanes x {sm_max:.0f} MHz (DESIGN.md §6.1)",
                    "algorithmic_instr_per_launch": DFMA_PER_TAU_POINT * w.n_tau * evaluated / max(args.steps, 1),
                    "launch_ms": 1e3 * kern_total / max(args.steps, 1),
                    "evaluated_moves_per_s": evaluated / kern_total,
                    "evaluated_fraction": evaluated / attempted, "accepted_fraction": accepted / attempted}
        try:
            # what the FP64 pipe delivers on the credited instructions alone (the tau loop with nothing else running,
            # `sail_microbench`): its three-operand DFMAs are operand-fetch bound (profiles/r02_sweep_pipe_bound.md)
            from paper_1609_07936_b200.binding import microbench
            mb = microbench(local_rank)
            loop_peak = mb["tau_loop_credited_per_clk_sm"] * 32 * num_sms * sm_max * 1e6
            roofline["credited_loop_alone"] = {"warp_instr_per_clk_sm": mb["tau_loop_credited_per_clk_sm"], "rate": loop_peak / 1e12,
                                               "unit": "T FP64 lane-instr/s", "frac_of_nominal": loop_peak / peak_nominal,
                                               "kernel_frac_of_it": achieved / loop_peak}
        except Exception as ex:  # supplementary only
            roofline["credited_loop_alone"] = {"error": repr(ex)}

        # the oracle on the host cores: rank 0, N = 1 only
        cpu_v, cores, sample = cpu_oracle_sample(w, target_s=args.cpu_seconds) if world == 1 else (None, None, None)
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
                "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                "dtype": "f64", "data": "synthetic",
                "config": config_dict(w, world),
                "anneals_per_s": world * args.steps / nb / total_s,
                "clocks": clocks, "e2e": e2e, "gpu_launches": launches, "roofline": roofline,
                "cpu_baseline": ({"value": cpu_v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample} if world == 1 else None),
                "chi2_final_median": float(np.median(chi2_final)),
                "build_defines": build_defines(),
                "history": HISTORY}
    s.close()
    del spectra_t, chi2_t, flush
    if rank == 0:
        if args.configs and world == 1:
            cfgs = {}
            for name in NAMES:
                if name == w.name and args.steps % nb == 0 and args.steps >= nb and not args.sweeps:
                    # the timed steps above were whole anneals of this configuration
                    cfgs[name] = {"workload": workload_string(w), "seconds_per_anneal": total_s * nb / args.steps,
                                  "anneals_per_s": args.steps / nb / total_s, "value": value, "unit": UNIT,
                                  "evaluated_fraction": roofline["evaluated_fraction"], "accepted_fraction": roofline["accepted_fraction"],
                                  "roofline_frac": roofline["frac_of_nominal"], "clocks": clocks, "note": "the headline run above"}
                    continue
                wc = wl.make(name)
                entry = whole_anneal(torch, Sail, wc, local_rank, peak_nominal, wc.rng_seed)
                if name == "noise":
                    entry["note"] = ("ONE of the 32 anneals of the noise sweep (eps = 1e-4); the whole sweep (4 eps x 8 anneals) is "
                                     "`python bench.py --noise-sweep`, profiles/r02_noise_sweep.json.txt")
                if name == "tiny":
                    cv, cc, cs = cpu_oracle_sample(wc, whole=True)
                    entry["cpu_oracle_whole_anneal"] = {"value": cv, "unit": UNIT, "cores": cc, "sample": cs}
                cfgs[name] = entry
            line["configs"] = cfgs
        if args.extra and world == 1:
            try:
                from paper_1609_07936_b200.binding import microbench
                line["microbench"] = microbench(local_rank)
                line["other_rows"] = extra_rows(torch, Sail, local_rank, peaks)
            except Exception as ex:  # supplementary only
                line["other_rows"] = {"error": repr(ex)}
        print(json.dumps(line))
    return 0


def main_noise_sweep(args):
    """BASELINE.json configs[3] as configured: relative noise eps in {1e-3, 1e-4, 1e-5, 1e-6} (seeds 4-7), 8 independent
    anneals each (Philox keys rng_seed + i), W = 16384.  Prints measured anneals/s (no extrapolation)."""
    import torch
    from paper_1609_07936_b200 import build
    build.build(defines=None if args.diag_defines else ())
    from paper_1609_07936_b200.binding import Sail
    peaks = measured_peaks()
    peak = torch.cuda.get_device_properties(0).multi_processor_count * FP64_LANES_PER_SM * (peaks.get("sm_max_mhz") or 1965.0) * 1e6
    out = {"workload": "noise sweep (BASELINE.json configs[3]): 4 eps x 8 anneals, W=16384, N_omega=1024, N_tau=256, 5000 sweeps, branching every 100",
           "anneals": []}
    t_all = time.perf_counter()
    for eps, nseed in wl.NOISE_SWEEP:
        w = wl.make("noise", eps=eps, noise_seed=nseed)
        for rep in range(args.noise_reps):
            e = whole_anneal(torch, Sail, w, 0, peak, w.rng_seed + rep)
            out["anneals"].append({"eps": eps, "rep": rep, "seconds": e["seconds_per_anneal"], "roofline_frac": e["roofline_frac"],
                                   "value": e["value"], "chi2_final_median": e["chi2_final_median"]})
    torch.cuda.synchronize()
    wall = time.perf_counter() - t_all
    n = len(out["anneals"])
    dev_s = sum(a["seconds"] for a in out["anneals"])
    out.update({"n_anneals": n, "wall_seconds_including_setup_and_warmup": wall, "device_seconds": dev_s, "anneals_per_s": n / dev_s,
                "attempted_moves_per_s": sum(a["value"] * a["seconds"] for a in out["anneals"]) / dev_s})
    print(json.dumps(out))
    return 0


def extra_rows(torch, Sail, dev_index, peaks):
    """Supplementary: the rows of SURVEY §8 a block of sweeps does not time on its own (A7 resync, A8 branching, f1-f4)
    against their own rooflines, on the 'stress' population."""
    out = {}
    w = wl.make("stress")
    s = Sail(w.omega, w.tau, w.F, w.sigma, max_walkers=w.W, device=dev_index)
    s.init_walkers(w.W, w.A, w.B, w.rng_seed)
    p = anneal_params(w)
    p["resync_every"] = 0

    def timed(fn, reps=1):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        e0.record()
        for _ in range(reps):
            fn()
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) * 1e-3 / reps

    s.anneal(w.schedule[:1], **p)                       # one sweep: a population with spread-out residues
    sm_max = peaks.get("sm_max_mhz", 1965.0)
    peak = torch.cuda.get_device_properties(dev_index).multi_processor_count * FP64_LANES_PER_SM * sm_max * 1e6
    hbm = peaks.get("hbm_gbs", 6553.3)
    s.resync()
    t_rs = timed(s.resync)
    flops = 2.0 * w.W * w.n_omega * w.n_tau
    out["stress_resync"] = {"seconds": t_rs, "tflops_fp64": flops / t_rs / 1e12,
                            "frac_of_fp64_alu_peak": flops / 2 / t_rs / peak}
    # f3 smoothing (Eq. 27-29): stencil + renormalisation kernel (HBM bound: the spectra once in, once out), then a resync
    s.smooth(0.02)
    t_sm = timed(lambda: s.smooth(0.02))
    sm_bytes = 16.0 * w.W * w.n_omega
    t_st = max(t_sm - t_rs, 1e-9)
    out["stress_smooth"] = {"seconds": t_sm, "stencil_seconds": t_st, "algorithmic_GB": sm_bytes / 1e9,
                            "stencil_GBps": sm_bytes / t_st / 1e9,
                            "frac_of_measured_hbm": sm_bytes / t_st / 1e9 / hbm,
                            "note": "stencil time = whole call minus the resync time measured above"}
    # one branching event per imprint strength, each on a fresh population (init + 1 sweep) so that the recipient
    # count belongs to the timed event itself; the kernels are warmed up on the old population first
    _, c2 = s.get(spectra=False)
    s.branch_async(float(np.std(c2)) * 0.5, 1.0)
    s.branch_async(float(np.std(c2)) * 0.5, 0.1)
    state = 8 * (w.n_omega + w.n_tau)
    for t_imp, key, streams in ((1.0, "stress_branch_t1", 2), (0.1, "stress_branch_t0.1", 3)):
        s.init_walkers(w.W, w.A, w.B, w.rng_seed)
        s.anneal(w.schedule[:1], **p)
        _, c2 = s.get(spectra=False)
        T = float(np.std(c2)) * 0.5
        box = {}
        l0 = s.launch_count()
        t_br = timed(lambda: box.update(info=s.branch(T, t_imp)[0]))
        n_rec = int(box["info"].n_recipients)
        # donor read + recipient write (+ recipient read when t < 1), plus chi^2 in and the fixed-point weights out
        algo_bytes = 16 * w.W + n_rec * state * streams
        out[key] = {"seconds": t_br, "recipients": n_rec, "algorithmic_GB": algo_bytes / 1e9, "kernel_launches": int(s.launch_count() - l0),
                    "achieved_GBps": algo_bytes / t_br / 1e9, "frac_of_measured_hbm": algo_bytes / t_br / 1e9 / hbm,
                    "note": "whole event + info read-back; donors with several recipients are re-read from L2"}
    # f2: the paper's branching step (a quarter of the walkers, t = 0.1): search of 1/T + the event itself;
    # f1: the residue statistics of the self-cooling schedule
    s.init_walkers(w.W, w.A, w.B, w.rng_seed)
    s.anneal(w.schedule[:1], **p)
    s.branch_fraction(0.25, 0.1)                        # warm-up on the same kind of population
    s.init_walkers(w.W, w.A, w.B, w.rng_seed)
    s.anneal(w.schedule[:1], **p)
    l0 = s.launch_count()
    box = {}
    t_bf = timed(lambda: box.update(r=s.branch_fraction(0.25, 0.1)))
    out["stress_branch_fraction_0.25"] = {"seconds": t_bf, "T_found": box["r"][0], "recipients": int(box["r"][1].n_recipients),
                                          "kernel_launches": int(s.launch_count() - l0)}
    out["stress_chi2_stats"] = {"seconds": timed(lambda: s.chi2_stats(), reps=5)}
    s.close()
    # f4: sweeps with the index-selection walk (2 steps) on Small, on the same screened batched kernel
    w2 = wl.make("small")
    s2 = Sail(w2.omega, w2.tau, w2.F, w2.sigma, max_walkers=w2.W, device=dev_index)
    p2 = anneal_params(w2)
    n2 = 100
    for L, key in ((0, "small_sweeps_walk0"), (2, "small_sweeps_walk2")):
        s2.init_walkers(w2.W, w2.A, w2.B, w2.rng_seed)
        s2.anneal(w2.schedule[:5], walk_length=L, **p2)
        _, ev0, _ = s2.stats()
        t_w = timed(lambda: s2.anneal(w2.schedule[5:5 + n2], walk_length=L, **p2))
        _, ev1, _ = s2.stats()
        out[key] = {"attempted_moves_per_s": w2.W * n2 * w2.n_omega / t_w, "seconds": t_w,
                    "evaluated_fraction": float((ev1 - ev0).sum()) / (w2.W * n2 * w2.n_omega),
                    "evaluated_moves_per_s": float((ev1 - ev0).sum()) / t_w,
                    "roofline_frac": DFMA_PER_TAU_POINT * w2.n_tau * float((ev1 - ev0).sum()) / t_w / peak}
    s2.close()
    return out


if __name__ == "__main__":
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="stress", choices=NAMES)
    ap.add_argument("--sweeps", type=int, default=0, help="override the number of sweeps (debug)")
    ap.add_argument("--cpu-seconds", type=float, default=12.0)
    ap.add_argument("--cpu-whole", action="store_true", help="--impl reference: time the oracle on the whole anneal of the workload, once")
    ap.add_argument("--e2e", type=int, default=-1, help="steps of the end-to-end (host buffers) run; -1 = as many as --steps, 0 = skip")
    ap.add_argument("--configs", type=int, default=1, help="also run one whole anneal of each BASELINE.json configuration (N=1 only)")
    ap.add_argument("--extra", type=int, default=1, help="also time resync / smoothing / branching / walk rows and the microbenchmarks (N=1 only)")
    ap.add_argument("--profile-sweeps", type=int, default=0, help="after the timed steps: re-init, anneal to --profile-at, then one launch of N sweeps (ncu target)")
    ap.add_argument("--profile-at", type=int, default=-1, help="sweep index of the --profile-sweeps launch (-1 = mid-anneal)")
    ap.add_argument("--selfcool", type=int, default=0, help="run N blocks of the paper's self-cooling protocol instead of the bench (supplementary)")
    ap.add_argument("--noise-sweep", action="store_true", help="run BASELINE.json configs[3] as configured (4 eps x --noise-reps anneals)")
    ap.add_argument("--noise-reps", type=int, default=8)
    ap.add_argument("--diag-defines", action="store_true",
                    help="time the library as it is on disk, with whatever -D flags it was built with (python -m paper_1609_07936_b200.build "
                         "--define ...); default: rebuild the product library (no defines) first.  The flags in force are in `build_defines`")
    a = ap.parse_args()
    if a.noise_sweep:
        sys.exit(main_noise_sweep(a))
    if a.selfcool > 0 and a.impl == "ours":
        sys.exit(main_selfcool(a))
    if a.gpus > 1 and "WORLD_SIZE" not in os.environ:
        sys.exit(spawn_ranks(a))
    sys.exit(main_reference(a) if a.impl == "reference" else main_ours(a))
