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


# ---- walker exchange (the DMC load balance of Alg. 1 L14) -------------------
# Off the hot path and not timed by bench.py: after branching, ranks hold different numbers of live walkers; whole
# walker states (Crowd.qmc_crowd_export_walkers / import_walkers: packed device buffers) move from ranks with a
# surplus to ranks with a deficit, point to point.  No collective touches the move / update path itself.

def balance_plan(counts):
    """Deterministic load-balance plan for per-rank live-walker counts: a list of (src_rank, dst_rank, n) transfers
    after which every rank holds floor(total / R) walkers, the first total % R ranks one more.  Every rank computes
    the same plan from the same all-gathered counts; surpluses are matched to deficits in rank order."""
    counts = [int(c) for c in counts]
    R, total = len(counts), sum(counts)
    assert R >= 1 and all(c >= 0 for c in counts)
    target = [total // R + (1 if r < total % R else 0) for r in range(R)]
    surplus = [[r, counts[r] - target[r]] for r in range(R) if counts[r] > target[r]]
    deficit = [[r, target[r] - counts[r]] for r in range(R) if counts[r] < target[r]]
    plan, i, j = [], 0, 0
    while i < len(surplus) and j < len(deficit):
        n = min(surplus[i][1], deficit[j][1])
        plan.append((surplus[i][0], deficit[j][0], n))
        surplus[i][1] -= n
        deficit[j][1] -= n
        if surplus[i][1] == 0:
            i += 1
        if deficit[j][1] == 0:
            j += 1
    return plan


def gather_counts(n_live: int, device="cpu"):
    """All ranks' live-walker counts (identity when not distributed)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return [int(n_live)]
    t = torch.zeros(dist.get_world_size(), dtype=torch.int64, device=device)
    t[dist.get_rank()] = int(n_live)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return [int(x) for x in t.tolist()]


def exchange_states(plan, rank: int, take, put, state_bytes: int, device="cpu"):
    """Run this rank's part of `plan`.  take(n) -> uint8 tensor [n, state_bytes] of n packed walker states leaving
    this rank (the caller chooses which and frees their slots); put(buf) receives a uint8 tensor [n, state_bytes].
    Sends and receives are posted together (isend / irecv) and waited for at the end."""
    import torch
    import torch.distributed as dist
    reqs, incoming = [], []
    for src, dst, n in plan:
        if n == 0 or src == dst:
            continue
        if rank == src:
            buf = take(n)
            assert buf.dtype == torch.uint8 and tuple(buf.shape) == (n, state_bytes)
            reqs.append(dist.isend(buf.contiguous(), dst))
        elif rank == dst:
            buf = torch.empty((n, state_bytes), dtype=torch.uint8, device=device)
            reqs.append(dist.irecv(buf, src))
            incoming.append(buf)
    for r in reqs:
        r.wait()
    for buf in incoming:
        put(buf)
    return sum(b.shape[0] for b in incoming)
