"""N>1 path on CPU: walker sharding and the scalar reductions bench.py uses, with
the gloo backend at world_size 2 (no collective on the data path)."""
import os
import socket

import numpy as np
import pytest
import torch.multiprocessing as mp

from paper_2602_05255_b200 import shard
from paper_2602_05255_b200 import workload as wl


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, q):
    import torch.distributed as dist

    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank),
                      WORLD_SIZE=str(world), LOCAL_RANK=str(rank))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    r, lr, ws = shard.env_rank()
    W = 6
    w0, w1 = shard.walker_range(r, ws, W)
    # each rank draws proposals for ITS global walker ids
    P, J, xi = wl.proposals(77, w1, 3, 16, 32, 2, walkers=range(w0, w1))
    shard.barrier()
    ms_max, = shard.reduce_scalars([10.0 + rank], "max")
    tot, = shard.reduce_scalars([float(W)], "sum")
    q.put((rank, w0, w1, P.tolist(), ms_max, tot))
    dist.destroy_process_group()


def test_two_rank_sharding_matches_single_process():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert [(r[1], r[2]) for r in res] == [(0, 6), (6, 12)]
    # trajectories depend on the global walker id only, not on the rank count
    P_all, _, _ = wl.proposals(77, 12, 3, 16, 32, 2)
    got = np.concatenate([np.array(r[3]) for r in res], axis=1)
    assert np.array_equal(got, P_all)
    assert all(r[4] == 11.0 for r in res)        # max over ranks
    assert all(r[5] == 12.0 for r in res)        # whole-job walker count


def test_split_and_range_helpers():
    assert shard.split_walkers(10, 3) == [(0, 4), (4, 7), (7, 10)]
    assert shard.split_walkers(0, 2) == [(0, 0), (0, 0)]
    assert shard.walker_range(3, 4, 5) == (15, 20)
    with pytest.raises(ValueError):
        shard.walker_range(4, 4, 5)
    assert shard.reduce_scalars([1.5, 2.0], "sum") == [1.5, 2.0]   # no process group: identity
