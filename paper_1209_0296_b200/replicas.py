"""N > 1: replicas only (BASELINE.json rules out sharding and collectives on the data path).

Every rank runs an independent lattice -- the workload's parameters with a rank-specific seed -- on its own
GPU.  The only communication is the bookkeeping of the measurement: the slowest rank's device time (MAX) and
the number of attempted updates all ranks made (SUM).  Host logic only; tested with gloo on CPU.
"""
from __future__ import annotations

import torch
import torch.distributed as dist

SEED_STRIDE = 4096   # workloads.seed_of: cfg*256 + variant < 4096 for cfg < 16, so rank seeds never collide


def rank_seed(seed: int, rank: int) -> int:
    """Seed of replica `rank`: rank 0 keeps the workload's seed (so N = 1 is the plain workload)."""
    return seed + SEED_STRIDE * rank


def aggregate(local_ms: float, local_updates: int, device="cpu") -> tuple[float, float, float]:
    """(max over ranks of the device time in ms, updates of all ranks, updates per second of the whole job)."""
    t = torch.tensor([float(local_ms)], dtype=torch.float64, device=device)
    u = torch.tensor([float(local_updates)], dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        dist.all_reduce(u, op=dist.ReduceOp.SUM)
    ms, upd = float(t.item()), float(u.item())
    return ms, upd, upd / (ms * 1e-3)
