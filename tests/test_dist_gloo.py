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
