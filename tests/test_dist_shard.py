"""N>1 host logic on CPU: two gloo ranks shard the pose list without overlap and agree on the max-over-ranks time."""
import os
import socket

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2408_12894_b200.shard import max_over_ranks, pose_index


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, n_poses, steps, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    mine = [pose_index(k, rank, world, n_poses) for k in range(steps)]
    gathered = [None] * world
    dist.all_gather_object(gathered, mine)
    t = max_over_ranks([10.0 + rank, 5.0 - rank], dist)
    dist.barrier()
    q.put((rank, mine, gathered, t))
    dist.destroy_process_group()


def test_two_ranks_shard_poses_and_reduce_time():
    world, n_poses, steps = 2, 200, 100
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, n_poses, steps, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = [q.get(timeout=120) for _ in range(world)]
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, mine, gathered, t in res:
        assert t == [11.0, 5.0]                       # max over ranks of (10+rank, 5-rank)
        flat = [x for g in gathered for x in g]
        assert sorted(flat) == list(range(n_poses))   # together: every pose exactly once
        assert set(gathered[0]).isdisjoint(gathered[1])


def test_single_process_is_identity():
    assert max_over_ranks([1.5, 2.5]) == [1.5, 2.5]
    assert [pose_index(k, 0, 1, 7) for k in range(9)] == [0, 1, 2, 3, 4, 5, 6, 0, 1]
