"""Multi-GPU plumbing (one process per GPU).  The SAIL hot path needs no data-path collective when the
anneal has no branching across ranks: walkers are independent Markov chains, so ranks run
independent replicas / walker shards ("scaling": "weak").  The only exchange is the timing reduction
(max over ranks) and the count of processed units — done with torch.distributed (nccl on GPUs, gloo in the
CPU tests)."""
from __future__ import annotations

import os


def env_world():
    return int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))


def init(backend: str):
    import torch.distributed as dist
    rank, local_rank, world = env_world()
    if world > 1 and not dist.is_initialized():
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29511")
        dist.init_process_group(backend=backend, rank=rank, world_size=world)
    return rank, local_rank, world


def rank_seed(base_seed: int, rank: int) -> int:
    """Philox key of a rank's replica: ranks draw disjoint streams (key differs in the high word)."""
    return (base_seed & 0xFFFFFFFF) | (((base_seed >> 32) + rank + 1) << 32) if rank else base_seed


def shard_walkers(W: int, rank: int, world: int):
    """Contiguous walker range of a rank: [lo, hi)."""
    base, rem = divmod(W, world)
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)


def reduce_timing(elapsed_s: float, units: float, device=None):
    """(max over ranks of elapsed, sum over ranks of units).  Works on nccl (device tensor) and gloo (cpu)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return elapsed_s, units
    t = torch.tensor([elapsed_s], dtype=torch.float64, device=device)
    u = torch.tensor([units], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), float(u.item())


def barrier(device=None):
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        if device is not None and str(device).startswith("cuda"):
            dist.barrier(device_ids=[int(str(device).split(":")[1])])
        else:
            dist.barrier()
