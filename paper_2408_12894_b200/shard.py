"""Multi-GPU plumbing: the path shards by camera pose -- frames are independent, the scene is replicated,
and no collective touches the data path ("replicas only").  torch.distributed is used for the barrier and for the
max-over-ranks time."""
from __future__ import annotations


def pose_index(step: int, rank: int, world: int, n_poses: int) -> int:
    """Pose rendered by `rank` at its step `step`: ranks interleave over the pose list (weak scaling: every rank
    does the same number of steps; together the ranks of one step cover `world` consecutive poses)."""
    return (rank + step * world) % n_poses


def max_over_ranks(values, dist=None, device=None):
    """Element-wise max of a list of floats over all ranks (identity without a process group)."""
    if dist is None or not dist.is_initialized():
        return list(values)
    import torch
    t = torch.tensor(list(values), dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(v) for v in t]
