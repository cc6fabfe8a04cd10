"""N>1 host logic on CPU: two gloo ranks shard the pose list without overlap and agree on the max-over-ranks time."""
import os
import socket

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2408_12894_b200.shard import RowShardedFrame, max_over_ranks, pose_index, rows_per_rank, tile_row_range


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


# ------------------------------------------------------------------ screen-space sharding (tile rows + one all-gather)

def _mock_rows(width, height):
    """Stands in for Renderer.render_rows on CPU: the strip of a synthetic image whose value names its (plane, row,
    column), written the way the library writes a strip ([3][rows][W], rows clipped to the image)."""
    def render_rows(tyb, tye, out):
        r0, r1 = 16 * tyb, min(height, 16 * tye)
        assert tuple(out.shape) == (3, r1 - r0, width)
        rows = torch.arange(r0, r1, dtype=torch.float32).view(1, -1, 1)
        cols = torch.arange(width, dtype=torch.float32).view(1, 1, -1)
        out.copy_(torch.arange(3, dtype=torch.float32).view(3, 1, 1) * 1e6 + rows * 1e3 + cols)
    return render_rows


def _expected(width, height):
    rows = torch.arange(height, dtype=torch.float32).view(1, -1, 1)
    cols = torch.arange(width, dtype=torch.float32).view(1, 1, -1)
    return torch.arange(3, dtype=torch.float32).view(3, 1, 1) * 1e6 + rows * 1e3 + cols


def _row_worker(rank, world, port, sizes, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ok = True
    for (w, h) in sizes:
        fr = RowShardedFrame(w, h, rank, world, torch.device("cpu"), dist)
        for _ in range(2):                                   # buffers are reused from frame to frame
            img = fr.render(_mock_rows(w, h))
        ok = ok and torch.equal(img, _expected(w, h))
    dist.barrier()
    q.put((rank, ok))
    dist.destroy_process_group()


def test_two_ranks_render_strips_and_gather_the_image():
    """Every rank really runs the sharding path end to end (strip -> all-gather -> stacked image) over gloo: image
    heights that split evenly, that leave the last strip clipped, and that leave the last rank without any row."""
    world = 2
    sizes = [(40, 64), (37, 50), (20, 16), (1920 // 8, 1080 // 4)]
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_row_worker, args=(r, world, port, sizes, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = [q.get(timeout=120) for _ in range(world)]
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert all(ok for _, ok in res)


def test_tile_row_ranges_partition_the_image():
    for h in (16, 17, 50, 545, 822, 1080):
        for world in (1, 2, 3, 4, 8):
            ty = (h + 15) // 16
            rng = [tile_row_range(r, world, h) for r in range(world)]
            assert rng[0][0] == 0 and rng[-1][1] == ty and all(a[1] == b[0] for a, b in zip(rng, rng[1:]))
            assert all(e - b <= rows_per_rank(h, world) for b, e in rng)
    fr = RowShardedFrame(33, 50, 0, 1, torch.device("cpu"))   # a single rank: no process group needed
    assert torch.equal(fr.render(_mock_rows(33, 50)), _expected(33, 50))
