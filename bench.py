#!/usr/bin/env python
"""bench.py — SAIL hot path on B200: attempted walker-moves/s, anneals/s and the roofline fraction.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload small]

A "step" is ONE WHOLE ANNEAL of the workload (BASELINE.json configs[1], "Small", by default): all sweeps of
the temperature schedule (proposal, positivity, Delta chi^2 over all tau, Metropolis, Eq. 30 — one persistent
sweep-kernel launch), any resyncs / branchings the config prescribes, and the final sail_get.  Walkers are
re-initialised (untimed) before every step.  `value` is measured with inputs resident in HBM (device-side
sail_get); `e2e` goes through the C ABI with HOST buffers (create from host arrays, schedule H2D, spectra
and chi^2 D2H into pinned memory) inside the timed region.

`--impl reference` times the CPU oracle (oracle/, as it stands) on the host cores on a bounded sample of the
same workload (this tier has no reference implementation to install).
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
FP64_LANES_PER_SM = 64          # DFMA lanes per SM per clock (4 sub-partitions x 16), see DESIGN.md §7
DFMA_PER_TAU_POINT = 5          # algorithmic FP64-pipe instructions per tau-point per evaluated move


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


# dram__bytes_read.sum + dram__bytes_write.sum of one sweep-kernel launch, from the committed ncu --set full capture
# (profiles/r01_sweep_small_full_metrics.txt): 12.06 MB + 3.07 MB for the whole 5000-sweep Small anneal
SWEEP_DRAM_BYTES_PER_LAUNCH = {("small", 5000): 15.13e6}


def anneal_params(w):
    return dict(eta=w.eta, amp_mode=1, amp_p=1.0, amp_m=2.0, y_min=1e-6, resync_every=w.resync_every)


# ------------------------------------------------------------------------------------------------
def run_protocol(s, w, torch, spectra_t=None, chi2_t=None, host_out=None):
    """One whole anneal on an initialised handle: sweeps (+ resync inside sail_anneal) + branching every
    branch_every sweeps + final sail_get.  Returns the CUDA events bracketing the sweep kernels."""
    p = anneal_params(w)
    ev = []
    done = 0
    n = w.n_sweeps
    while done < n:
        chunk = min(w.branch_every, n - done) if w.branch_every else n
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        s.anneal(w.schedule[done:done + chunk], **p)
        e1.record()
        ev.append((e0, e1))
        done += chunk
        if w.branch_every and done % w.branch_every == 0:
            s.branch_async(float(w.schedule[done - 1]), w.t_imprint)
    if host_out is not None:
        s.get_into(*host_out)
    else:
        s.get_device(spectra_t, chi2_t)
    return ev


def cpu_oracle_sample(w, target_s=12.0, seed=0x5A11):
    """Oracle (as it stands) on the host cores, on a bounded sample: a subset of walkers over the first
    sweeps of the schedule.  Returns (moves/s, cores, description)."""
    import oracle
    cores = oracle.num_threads()
    Ws = max(cores * 8, 64)
    o = oracle.Oracle(w.omega, w.tau, w.F, w.sigma, w.A, w.B, w.eta, seed)
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
    vals = []
    for _ in range(args.warmup):
        cpu_oracle_sample(w, target_s=1.0)
    t_per = max(2.0, min(20.0, 60.0 / max(args.steps, 1)))
    for _ in range(args.steps):
        v, cores, sample = cpu_oracle_sample(w, target_s=t_per)
        vals.append(v)
    value = float(np.mean(vals))
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * w.attempted_moves() / value,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"{w.name}: N_omega={w.n_omega}, N_tau={w.n_tau}, W={w.W}, sweeps={w.n_sweeps}",
                       "note": "CPU oracle on host cores; ms_per_step extrapolated from the bounded sample"},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))
    return 0


def main_selfcool(args):
    """Supplementary: the paper's own protocol (self-cooling, blocks of 100 sweeps, smoothing, a quarter of the walkers
    branched with t = 0.1, strength following the acceptance rate) on the chosen workload; prints the trajectory."""
    import torch
    from paper_1609_07936_b200 import build
    build.build()
    from paper_1609_07936_b200.binding import Sail
    w = wl.make(args.workload)
    s = Sail(w.omega, w.tau, w.F, w.sigma, max_walkers=w.W)
    s.init_walkers(w.W, w.A, w.B, w.rng_seed)
    nb, k = args.selfcool, 100
    kw = dict(n_boil=max(1, nb // 10), n_ramp=max(1, nb // 5), eta=w.eta, t_imprint=0.1, smooth_s=0.01, branch_fraction=0.25,
              adapt=True, freeze_rate=0.5)
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    T, ave, mn = s.anneal_selfcool(nb, k, **kw)
    torch.cuda.synchronize()
    dt = time.perf_counter() - t0
    mn_end, ave_end = s.chi2_stats()
    acc, ev, _ = s.stats()
    print(json.dumps({"protocol": "self-cooling (sail_anneal_selfcool)", "workload": w.name, "blocks": nb, "sweeps_per_block": k,
                      "parameters": {a: b for a, b in kw.items() if a != "eta"}, "seconds": dt,
                      "attempted_moves_per_s": w.W * nb * k * w.n_omega / dt, "accepted_fraction": float(acc.sum()) / (w.W * nb * k * w.n_omega),
                      "T": [float(x) for x in T], "chi2_ave": [float(x) for x in ave], "chi2_min": [float(x) for x in mn],
                      "chi2_ave_end": ave_end, "chi2_min_end": mn_end, "n_tau": w.n_tau}))
    s.close()
    return 0


def main_ours(args):
    import torch
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (no CPU fallback); use --impl reference for the oracle")
    from paper_1609_07936_b200 import build
    build.build()
    from paper_1609_07936_b200.binding import Sail, measure_fp64_peak

    rank, local_rank, world = sdist.init("nccl")
    torch.cuda.set_device(local_rank)
    dev = f"cuda:{local_rank}"
    w = wl.make(args.workload)
    if args.sweeps:
        w = w.scaled(n_sweeps=args.sweeps)
    seed = sdist.rank_seed(w.rng_seed, rank)          # every rank anneals an independent replica (weak scaling)
    peaks = measured_peaks()

    spectra_t = torch.empty((w.W, w.n_omega), dtype=torch.float64, device=dev)
    chi2_t = torch.empty(w.W, dtype=torch.float64, device=dev)
    flush = torch.empty(256 * 1024 * 1024 // 4, dtype=torch.float32, device=dev)   # > L2 (126 MB)
    s = Sail(w.omega, w.tau, w.F, w.sigma, max_walkers=w.W, device=local_rank)

    def one_step(timed):
        s.init_walkers(w.W, w.A, w.B, seed)            # untimed set-up of the step (A1)
        flush.zero_()                                   # L2 flush between timed iterations
        torch.cuda.synchronize()
        l0 = s.launch_count()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        kev = run_protocol(s, w, torch, spectra_t, chi2_t)
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) * 1e-3, sum(a.elapsed_time(b) for a, b in kev) * 1e-3, len(kev), s.launch_count() - l0

    for _ in range(args.warmup):
        one_step(False)
    sampler = ClockSampler(local_rank)
    sdist.barrier(dev)
    torch.cuda.synchronize()
    sampler.start()
    step_s, kern_s, n_sweep_launches, launches = [], [], 0, 0
    for _ in range(args.steps):
        t, k, nl, lc = one_step(True)
        step_s.append(t); kern_s.append(k); n_sweep_launches += nl; launches += lc
    torch.cuda.synchronize()
    sdist.barrier(dev)
    clocks = sampler.stop()
    acc, ev, _ = s.stats()                              # of the last step (deterministic per step)
    evaluated = float(ev.sum())
    accepted = float(acc.sum())
    chi2_final = chi2_t.cpu().numpy()

    total_s, total_moves = sdist.reduce_timing(float(np.sum(step_s)), float(w.attempted_moves() * args.steps), dev)
    value = total_moves / total_s
    ms_per_step = 1e3 * total_s / args.steps

    line = None
    if rank == 0:
        # ---- roofline of the dominant kernel (the sweep kernel): FP64 ALU bound ----------------------
        sm_max = peaks.get("sm_max_mhz") or clocks.get("sm_max_mhz") or 1965.0
        num_sms = torch.cuda.get_device_properties(local_rank).multi_processor_count
        peak_nominal = num_sms * FP64_LANES_PER_SM * sm_max * 1e6
        dfma_measured = measure_fp64_peak(local_rank)
        kern_total = float(np.sum(kern_s))
        algo_instr_per_launch = DFMA_PER_TAU_POINT * w.n_tau * evaluated / max(n_sweep_launches / args.steps, 1)
        achieved = DFMA_PER_TAU_POINT * w.n_tau * evaluated * args.steps / kern_total
        roofline = {"bound": "alu", "kernel": "sail::sweep_kernel", "achieved": achieved / 1e12, "peak": peak_nominal / 1e12,
                    "unit": "T FP64 lane-instr/s", "frac": achieved / peak_nominal, "traffic": SWEEP_DRAM_BYTES_PER_LAUNCH.get((w.name, w.n_sweeps)),
                    "peak_source": f"derived: {num_sms} SMs x {FP64_LANES_PER_SM} FP64 lanes x {sm_max:.0f} MHz (DESIGN.md §7)",
                    "peak_measured_dfma": dfma_measured / 1e12, "frac_of_measured_dfma": achieved / dfma_measured,
                    "algorithmic_instr_per_launch": algo_instr_per_launch,
                    "launch_ms": 1e3 * kern_total / max(n_sweep_launches, 1),
                    "evaluated_moves_per_s": evaluated * args.steps / kern_total,
                    "evaluated_fraction": evaluated / w.attempted_moves(), "accepted_fraction": accepted / w.attempted_moves()}

        # ---- end to end through the C ABI with host buffers --------------------------------------------
        host_sp = torch.empty((w.W, w.n_omega), dtype=torch.float64).pin_memory().numpy()
        host_c2 = torch.empty(w.W, dtype=torch.float64).pin_memory().numpy()
        e2e_s = []
        for it in range(1 + min(args.steps, 3)):
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            s2 = Sail(w.omega, w.tau, w.F, w.sigma, max_walkers=w.W, device=local_rank)     # H2D of the problem
            s2.init_walkers(w.W, w.A, w.B, seed)
            run_protocol(s2, w, torch, host_out=(host_sp, host_c2))                        # schedule H2D, results D2H
            torch.cuda.synchronize()
            dt = time.perf_counter() - t0
            s2.close()
            if it:
                e2e_s.append(dt)
        assert np.array_equal(host_c2, chi2_final), "e2e run is not bit-identical to the device-resident run"
        h2d = 8 * (w.n_omega + 3 * w.n_tau + w.n_sweeps)
        d2h = 8 * (w.W * w.n_omega + w.W)
        e2e = {"value": w.attempted_moves() / float(np.mean(e2e_s)), "unit": UNIT, "h2d_bytes_per_step": h2d,
               "d2h_bytes_per_step": d2h, "anneals_per_s": 1.0 / float(np.mean(e2e_s)),
               "includes": "sail_create + sail_init_walkers + anneal protocol + sail_get to pinned host + sail_destroy"}

        cpu_v, cores, sample = cpu_oracle_sample(w, target_s=args.cpu_seconds)
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
                "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                "dtype": "f64", "data": "synthetic",
                "config": {"workload": f"{w.name} (BASELINE.json configs[{['tiny', 'small', 'branching', 'noise', 'stress'].index(w.name)}]): N_omega={w.n_omega}, N_tau={w.n_tau}, W={w.W}, "
                                       f"sweeps={w.n_sweeps}, T {w.t0}->{w.t1} geometric, eps={w.eps}",
                           "step": "one whole anneal (all sweeps + final sail_get), walkers re-initialised untimed",
                           "parallelism": f"{world} independent replica(s), one per GPU", "l2": "flushed between steps (256 MiB write)",
                           "attempted_moves_per_step": w.attempted_moves()},
                "anneals_per_s": world * args.steps / total_s,
                "clocks": clocks, "e2e": e2e, "gpu_launches": launches, "roofline": roofline,
                "cpu_baseline": {"value": cpu_v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
                "chi2_final_median": float(np.median(chi2_final))}
        if args.extra and world == 1:
            try:
                from paper_1609_07936_b200.binding import microbench
                line["microbench"] = microbench(local_rank)
                line["other_workloads"] = extra_workloads(torch, Sail, local_rank, peaks)
            except Exception as ex:  # supplementary only
                line["other_workloads"] = {"error": repr(ex)}
        print(json.dumps(line))
    s.close()
    return 0


def extra_workloads(torch, Sail, dev_index, peaks):
    """Supplementary: one block of the 'stress' config (sweeps + resync + imprinted branching) to time the
    rows the Small anneal does not contain (A7 resync, A8 branching) against their own rooflines."""
    out = {}
    w = wl.make("stress")
    n_sw = 4
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

    s.anneal(w.schedule[:1], **p)                       # warm-up
    acc0, ev0, _ = s.stats()
    t_sw = timed(lambda: s.anneal(w.schedule[1:1 + n_sw], **p))
    acc1, ev1, _ = s.stats()
    evaluated = float((ev1 - ev0).sum())
    sm_max = peaks.get("sm_max_mhz", 1965.0)
    peak = torch.cuda.get_device_properties(dev_index).multi_processor_count * FP64_LANES_PER_SM * sm_max * 1e6
    out["stress_sweeps"] = {"workload": f"stress: N_omega={w.n_omega}, N_tau={w.n_tau}, W={w.W}, {n_sw} sweeps",
                            "attempted_moves_per_s": w.W * n_sw * w.n_omega / t_sw, "seconds": t_sw,
                            "evaluated_fraction": evaluated / (w.W * n_sw * w.n_omega),
                            "roofline_frac": DFMA_PER_TAU_POINT * w.n_tau * evaluated / t_sw / peak}
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
                            "frac_of_measured_hbm": sm_bytes / t_st / 1e9 / peaks.get("hbm_gbs", 6553.3),
                            "note": "stencil time = whole call minus the resync time measured above"}
    # one branching event per imprint strength, each on a fresh population (init + 1 sweep) so that the recipient
    # count belongs to the timed event itself; the kernels are warmed up on the old population first
    _, c2 = s.get(spectra=False)
    s.branch_async(float(np.std(c2)) * 0.5, 1.0)
    s.branch_async(float(np.std(c2)) * 0.5, 0.1)
    state = 8 * (w.n_omega + w.n_tau)
    hbm = peaks.get("hbm_gbs", 6553.3)
    for t_imp, key, streams in ((1.0, "stress_branch_t1", 2), (0.1, "stress_branch_t0.1", 3)):
        s.init_walkers(w.W, w.A, w.B, w.rng_seed)
        s.anneal(w.schedule[:1], **p)
        _, c2 = s.get(spectra=False)
        T = float(np.std(c2)) * 0.5
        box = {}
        t_br = timed(lambda: box.update(info=s.branch(T, t_imp)[0]))
        n_rec = int(box["info"].n_recipients)
        # donor read + recipient write (+ recipient read when t < 1), plus chi^2 in and the fixed-point weights out
        algo_bytes = 16 * w.W + n_rec * state * streams
        out[key] = {"seconds": t_br, "recipients": n_rec, "algorithmic_GB": algo_bytes / 1e9,
                    "achieved_GBps": algo_bytes / t_br / 1e9, "frac_of_measured_hbm": algo_bytes / t_br / 1e9 / hbm,
                    "note": "whole event (12 launches + info read-back); donors with several recipients are re-read from L2"}
    # f2: the paper's branching step (a quarter of the walkers, t = 0.1): search of 1/T (one multiplier chain and one
    # 8-byte read-back per trial) + the event itself; f1: the two-kernel residue statistics of the self-cooling schedule
    s.init_walkers(w.W, w.A, w.B, w.rng_seed)
    s.anneal(w.schedule[:1], **p)
    l0 = s.launch_count()
    box = {}
    t_bf = timed(lambda: box.update(r=s.branch_fraction(0.25, 0.1)))
    out["stress_branch_fraction_0.25"] = {"seconds": t_bf, "T_found": box["r"][0], "recipients": int(box["r"][1].n_recipients),
                                          "kernel_launches": int(s.launch_count() - l0)}
    out["stress_chi2_stats"] = {"seconds": timed(lambda: s.chi2_stats(), reps=5)}
    s.close()
    # f4: sweeps with the index-selection walk (2 steps) on Small; it runs on the plain kernel (state-dependent proposals)
    w2 = wl.make("small")
    s2 = Sail(w2.omega, w2.tau, w2.F, w2.sigma, max_walkers=w2.W, device=dev_index)
    s2.init_walkers(w2.W, w2.A, w2.B, w2.rng_seed)
    p2 = anneal_params(w2)
    s2.anneal(w2.schedule[:5], walk_length=2, **p2)
    _, ev0, _ = s2.stats()
    n2 = 100
    t_w = timed(lambda: s2.anneal(w2.schedule[5:5 + n2], walk_length=2, **p2))
    _, ev1, _ = s2.stats()
    out["small_sweeps_walk2"] = {"attempted_moves_per_s": w2.W * n2 * w2.n_omega / t_w, "seconds": t_w,
                                 "evaluated_fraction": float((ev1 - ev0).sum()) / (w2.W * n2 * w2.n_omega),
                                 "roofline_frac": DFMA_PER_TAU_POINT * w2.n_tau * float((ev1 - ev0).sum()) / t_w / peak}
    s2.close()
    return out


if __name__ == "__main__":
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="small", choices=["tiny", "small", "branching", "noise", "stress"])
    ap.add_argument("--sweeps", type=int, default=0, help="override the number of sweeps (debug)")
    ap.add_argument("--cpu-seconds", type=float, default=12.0)
    ap.add_argument("--extra", type=int, default=1, help="also time a block of the stress config (N=1 only)")
    ap.add_argument("--selfcool", type=int, default=0, help="run N blocks of the paper's self-cooling protocol instead of the bench (supplementary)")
    a = ap.parse_args()
    if a.selfcool > 0 and a.impl == "ours":
        sys.exit(main_selfcool(a))
    sys.exit(main_reference(a) if a.impl == "reference" else main_ours(a))
