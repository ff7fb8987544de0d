"""sail_chi2_stats_static — population statistics for callers that may not allocate device memory.

Who needs it: a thread that watches a running anneal (progress monitor, stopping rule) works on a COPY of the
residues, because the handle and its workspace belong to the annealing thread; and it cannot call cudaMalloc /
cudaFree, which wait for the whole device — behind a sweep kernel that runs for seconds.  The entry point therefore
keeps its per-CTA partial results in ONE fixed 4 KB array per GPU that is part of the library image, shared by all
calls and never cleared.  What is checked here:
  * CPU: sizes beyond SAIL_STATS_STATIC_MAX_W (and NULL pointers) are refused with a clear message before the device
    is touched;
  * GPU: two calls in a row — a large population, then a small one that uses only a few slots of the array while the
    rest still holds the first call's partial results — each give what sail_chi2_stats (scratch in the handle's
    workspace) gives on the same residues, to the tolerance tests/test_gpu_parity.py uses for these statistics
    (minimum identical, mean to 1e-13 relative).

The file name sorts after every other test file on purpose: `pytest -x` stops at the first failure, and a failure
here must not hide the parity tests.  The GPU test runs alone in a fresh process (where its first call also performs
the per-device set-up) as well as after the other tests.
"""
import ctypes as C

import numpy as np
import pytest

from paper_1609_07936_b200 import workloads as wl

SEED = 0x5A11_0000_0000_0077


def test_sizes_beyond_the_fixed_scratch_are_refused_on_the_host():
    from paper_1609_07936_b200 import binding, build
    build.build(defines=())
    L = binding.lib()
    dummy = C.c_void_p(256)                                   # never dereferenced: the size check comes first
    too_many = binding.STATS_STATIC_MAX_W + 1
    assert L.sail_chi2_stats_static(0, None, dummy, too_many, dummy) == binding.SAIL_ERR_ARG
    msg = L.sail_last_error(None).decode()
    assert str(binding.STATS_STATIC_MAX_W) in msg and "SAIL_STATS_STATIC_MAX_W" in msg and "sail_chi2_stats" in msg
    assert L.sail_chi2_stats_static(0, None, dummy, 0, dummy) == binding.SAIL_ERR_ARG
    assert L.sail_chi2_stats_static(0, None, None, 8, dummy) == binding.SAIL_ERR_ARG
    assert L.sail_chi2_stats_static(0, None, dummy, 8, None) == binding.SAIL_ERR_ARG
    assert b"NULL" in L.sail_last_error(None)


@pytest.mark.gpu
def test_static_scratch_statistics_match_the_workspace_path_on_two_calls_in_a_row():
    import torch
    from paper_1609_07936_b200 import binding

    w = wl.make("tiny", simpson_intervals=20_000)
    W_big, W_small = 70_001, 301                              # 256 CTAs with a ragged tail, then 2 CTAs
    s = binding.Sail(w.omega, w.tau, w.F, w.sigma, max_walkers=W_big)
    out = torch.full((2,), float("nan"), dtype=torch.float64, device="cuda:0")
    chi2_t = torch.empty(W_big, dtype=torch.float64, device="cuda:0")
    for call, W in enumerate((W_big, W_small)):
        s.init_walkers(W, w.A, w.B, SEED + call)
        s.anneal(np.full(3, 1e6), w.eta)                      # hot sweeps: every walker ends at its own residue
        want_min, want_mean = s.chi2_stats()                  # existing path: partial results in the handle's workspace
        s.get_device(chi2_t=chi2_t)                           # the monitor's copy of the residues (first W entries)
        binding.chi2_stats_static(chi2_t, out, n=W)           # no handle, no allocation; same stream as the copy
        got_min, got_mean = out.cpu().numpy()
        c2 = chi2_t[:W].cpu().numpy()
        assert np.unique(c2).size > W // 2                    # the statistics are not those of a constant array
        assert got_min == want_min == c2.min()
        assert abs(got_mean - want_mean) <= 1e-13 * abs(want_mean)
        assert abs(got_mean - c2.mean()) <= 1e-13 * abs(c2.mean())
    s.close()
