"""Multi-GPU host logic on CPU: world_size-2 gloo run of the sharding / aggregation helpers that
bench.py uses under torchrun (walkers shard, no data-path collective)."""
import os
import socket

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world),
                      LOCAL_RANK=str(rank))
    from paper_2209_14487_b200 import dist as qd
    assert qd.env_world() == (rank, rank, world)
    qd.init("gloo")
    assert dist.is_initialized() and dist.get_world_size() == world
    id0, cnt = qd.walker_slice(rank, world, 256)
    qd.barrier()
    # rank r "took" (10 + 5 r) ms and processed cnt * 768 moves, accepted 100 (r + 1)
    ms, (moves, acc) = qd.reduce_job(10.0 + 5.0 * rank, [cnt * 768, 100 * (rank + 1)])
    out[rank] = (id0, cnt, ms, moves, acc)
    dist.destroy_process_group()


def test_walker_sharding_and_reduction_world2():
    world, port = 2, _free_port()
    with mp.Manager() as mgr:
        out = mgr.dict()
        mp.spawn(_worker, args=(world, port, out), nprocs=world, join=True)
        res = dict(out)
    assert res[0][:2] == (0, 256) and res[1][:2] == (256, 256)      # disjoint global walker ids
    for r in range(world):
        _, _, ms, moves, acc = res[r]
        assert ms == 15.0                                           # max over ranks
        assert moves == 2 * 256 * 768 and acc == 300                # sums over ranks


def test_single_process_is_identity():
    from paper_2209_14487_b200 import dist as qd
    assert qd.walker_slice(0, 1, 64) == (0, 64)
    assert qd.reduce_job(3.5, [7, 9]) == (3.5, [7, 9])
    with pytest.raises(AssertionError):
        qd.walker_slice(2, 2, 64)


# ---- walker exchange (DMC load balance, Alg. 1 L14 / PAPER.md:66): plan and point-to-point transport ----------
def test_balance_plan_properties():
    from paper_2209_14487_b200 import dist as qd
    import random
    rnd = random.Random(7)
    cases = [[5], [4, 4], [7, 1], [0, 9], [3, 3, 3, 11], [10, 0, 0, 0, 1]] + \
            [[rnd.randrange(0, 40) for _ in range(rnd.randrange(1, 9))] for _ in range(200)]
    for counts in cases:
        plan = qd.balance_plan(counts)
        after = list(counts)
        for src, dst, n in plan:
            assert src != dst and n > 0
            assert counts[src] > counts[dst]          # walkers only flow from richer to poorer ranks
            after[src] -= n
            after[dst] += n
        R, total = len(counts), sum(counts)
        assert after == [total // R + (1 if r < total % R else 0) for r in range(R)]
        assert sum(n for _, _, n in plan) == sum(max(0, c - a) for c, a in zip(counts, after))   # minimal traffic
    assert qd.balance_plan([4, 4]) == []
    assert qd.balance_plan([7, 1]) == [(0, 1, 3)]


def _exchange_worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world),
                      LOCAL_RANK=str(rank))
    from paper_2209_14487_b200 import dist as qd
    qd.init("gloo")
    nbytes = 48
    # rank 0 holds 7 live walkers, rank 1 holds 2; a "state" is 48 bytes tagged with (rank, walker)
    live = {0: 7, 1: 2}[rank]
    states = [torch.full((nbytes,), 16 * rank + i, dtype=torch.uint8) for i in range(live)]
    counts = qd.gather_counts(live)
    plan = qd.balance_plan(counts)

    def take(n):
        return torch.stack([states.pop() for _ in range(n)])

    def put(buf):
        states.extend(list(buf))

    got = qd.exchange_states(plan, rank, take, put, nbytes)
    out[rank] = (counts, plan, got, sorted(int(s[0]) for s in states), all(bool((s == s[0]).all()) for s in states))
    dist.destroy_process_group()


def test_walker_exchange_world2():
    world, port = 2, _free_port()
    with mp.Manager() as mgr:
        out = mgr.dict()
        mp.spawn(_exchange_worker, args=(world, port, out), nprocs=world, join=True)
        res = dict(out)
    for r in range(world):
        assert res[r][0] == [7, 2] and res[r][1] == [(0, 1, 2)]     # same counts and plan on every rank
        assert res[r][4]                                            # every state arrived intact
    assert res[0][2] == 0 and res[1][2] == 2
    assert res[0][3] == [0, 1, 2, 3, 4]                             # rank 0 kept five, sent its last two
    assert res[1][3] == [5, 6, 16, 17]                              # rank 1 has its own two plus walkers 5, 6 of rank 0
