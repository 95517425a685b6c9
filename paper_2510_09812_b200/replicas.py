"""Replica bookkeeping for `bench.py --gpus N` (the path does not shard -- replicas only).

Each rank steps its own independent replica; there is no collective on the data path.  The only communication is the
timing contract: a barrier on both sides of the timed region and the MAX over ranks of the per-rank device time.
"""
from __future__ import annotations

import os


def world_info():
    return int(os.environ.get("WORLD_SIZE", "1")), int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0"))


def barrier(dist=None):
    if dist is not None and dist.is_initialized() and dist.get_world_size() > 1:
        dist.barrier()


def aggregate(steps_per_rank: int, local_ms: float, dist=None, device=None):
    """Whole-job throughput: (replicas * steps) / max-over-ranks time.  Returns (world, max_ms, steps_per_second)."""
    world = 1
    max_ms = float(local_ms)
    if dist is not None and dist.is_initialized() and dist.get_world_size() > 1:
        import torch
        world = dist.get_world_size()
        t = torch.tensor([local_ms], dtype=torch.float64, device=device if device is not None else "cpu")
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        max_ms = float(t.item())
    return world, max_ms, world * steps_per_rank / (max_ms * 1e-3)
