"""Multi-GPU plumbing: the path shards over walkers with NO data-path
collective (walkers are independent); each rank owns one crowd and its slice of the
global walker ids, so Philox streams stay global (reading C7).  torch.distributed is used only for
the barrier, the max-over-ranks of the device time and the sum of the counters."""
from __future__ import annotations

import os


def env_world():
    """(rank, local_rank, world_size) from the torchrun environment; (0, 0, 1) when absent."""
    return (int(os.environ.get("RANK", 0)), int(os.environ.get("LOCAL_RANK", 0)),
            int(os.environ.get("WORLD_SIZE", 1)))


def walker_slice(rank: int, world: int, walkers_per_rank: int):
    """Weak scaling: every rank advances `walkers_per_rank` walkers; returns (walker_id0, count)."""
    assert 0 <= rank < world and walkers_per_rank >= 1
    return rank * walkers_per_rank, walkers_per_rank


def init(backend: str):
    import torch.distributed as dist
    if dist.is_available() and not dist.is_initialized() and int(os.environ.get("WORLD_SIZE", 1)) > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group(backend=backend)
    return dist


def barrier():
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized():
        dist.barrier()


def reduce_job(elapsed_ms: float, counters, device="cpu"):
    """Max over ranks of the device time, sum over ranks of integer counters.
    Returns (max_ms, [summed counters]); identity when not distributed."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return float(elapsed_ms), [int(c) for c in counters]
    t = torch.tensor([elapsed_ms], dtype=torch.float64, device=device)
    c = torch.tensor([int(x) for x in counters], dtype=torch.int64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(c, op=dist.ReduceOp.SUM)
    return float(t.item()), [int(x) for x in c.tolist()]
