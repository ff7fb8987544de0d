"""Host-side logic of the multi-GPU (one process per GPU) path, exercised with gloo at world_size 2 on CPU:
walker sharding, per-rank Philox keys, and the max-over-ranks timing / sum-over-ranks unit reduction that
bench.py uses.  The SAIL hot path has no data-path collective when ranks run independent replicas
(DESIGN.md §9)."""
import os
import socket
import subprocess
import sys

import numpy as np

from paper_1609_07936_b200 import distributed as sdist

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import os, sys, json
sys.path.insert(0, {root!r})
import numpy as np
from paper_1609_07936_b200 import distributed as sdist
import oracle
from paper_1609_07936_b200 import workloads as wl
rank, local_rank, world = sdist.init("gloo")
assert world == 2
lo, hi = sdist.shard_walkers(10, rank, world)
seed = sdist.rank_seed(0x5A11, rank)
# each rank anneals its own independent replica of a tiny problem with the oracle (CPU stand-in for the GPU rank)
w = wl.make("tiny", simpson_intervals=2000)
o = oracle.Oracle(w.omega, w.tau, w.F, w.sigma, w.A, w.B, w.eta, seed)
o.init_walkers(4)
o.anneal(w.schedule[:3])
elapsed = 1.0 + rank          # fake per-rank device time
units = float(4 * 3 * w.n_omega)
sdist.barrier()
t, u = sdist.reduce_timing(elapsed, units)
print(json.dumps(dict(rank=rank, lo=lo, hi=hi, seed=seed, t=t, u=u, chi2=float(o.chi2.sum()))))
"""


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def test_shard_walkers_partitions_exactly():
    for W, world in [(10, 2), (7, 3), (4096, 8), (5, 8)]:
        parts = [sdist.shard_walkers(W, r, world) for r in range(world)]
        assert parts[0][0] == 0 and parts[-1][1] == W
        assert all(parts[i][1] == parts[i + 1][0] for i in range(world - 1))
        sizes = [b - a for a, b in parts]
        assert max(sizes) - min(sizes) <= 1


def test_rank_seeds_are_distinct_keys():
    seeds = {sdist.rank_seed(0x5A11, r) for r in range(8)}
    assert len(seeds) == 8 and sdist.rank_seed(0x5A11, 0) == 0x5A11
    assert all(s & 0xFFFFFFFF == 0x5A11 for s in seeds)


def test_two_rank_gloo_timing_reduction():
    import json
    port = _free_port()
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port), OMP_NUM_THREADS="2")
        procs.append(subprocess.Popen([sys.executable, "-c", WORKER.format(root=ROOT)], env=env,
                                      stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True))
    outs = []
    for p in procs:
        out, err = p.communicate(timeout=180)
        assert p.returncode == 0, err[-2000:]
        outs.append(json.loads(out.strip().splitlines()[-1]))
    outs.sort(key=lambda d: d["rank"])
    assert [o["t"] for o in outs] == [2.0, 2.0]                 # max over ranks
    assert outs[0]["u"] == outs[1]["u"] == 2 * 4 * 3 * 64       # sum over ranks
    assert (outs[0]["lo"], outs[0]["hi"], outs[1]["lo"], outs[1]["hi"]) == (0, 5, 5, 10)
    assert outs[0]["seed"] != outs[1]["seed"]
    assert outs[0]["chi2"] != outs[1]["chi2"]                   # different keys -> different chains


def test_single_process_reduce_is_identity():
    assert sdist.reduce_timing(1.5, 10.0) == (1.5, 10.0)
