"""Multi-GPU plumbing.  One process per GPU; torch.distributed carries the barrier, the
max-over-ranks time and -- in screen-space sharding -- ONE all-gather of image strips per frame.  No arithmetic of the
method lives here: a strip is rendered by the library (flod_render_rows), this module decides which rows a rank owns and
stacks the gathered strips.

Two ways to shard:
  * poses   ("replicas"): frames are independent, every rank holds the whole scene and renders its own poses; no
            collective touches the data path (weak scaling);
  * rows    every rank renders the same pose's strip of tile rows [ty_begin, ty_end) -- it culls the Gaussians to its strip,
            lists, orders and blends only its own tiles -- and one all-gather (NCCL over NVLink / NVSwitch; 6-25 MB per
            frame) assembles the image on every rank (strong scaling; for the 1920x1080 / 15 M-Gaussian config, where one
            frame is large enough to split: the long trajectories of P:699-707).
"""
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


def rows_per_rank(height: int, world: int, tile: int = 16) -> int:
    """Tile rows every rank owns: the same number for all (the all-gather wants equal pieces); the last ranks' strips
    may reach past the image and are clipped."""
    ty = (height + tile - 1) // tile
    return (ty + world - 1) // world


def tile_row_range(rank: int, world: int, height: int, tile: int = 16):
    """[ty_begin, ty_end) of `rank`: consecutive strips of rows_per_rank tile rows, clipped to the image."""
    ty = (height + tile - 1) // tile
    per = rows_per_rank(height, world, tile)
    return min(rank * per, ty), min((rank + 1) * per, ty)


class RowShardedFrame:
    """Buffers and the collective of screen-space sharding for one image size.  `render_rows(ty_begin, ty_end, out)` is
    the library call (Renderer.render_rows bound to a camera and mode) that writes [3][rows][W] into `out`."""

    def __init__(self, width: int, height: int, rank: int, world: int, device, dist=None, tile: int = 16):
        import torch
        self.torch, self.dist = torch, dist
        self.W, self.H, self.rank, self.world, self.tile = width, height, rank, world, tile
        self.per = rows_per_rank(height, world, tile)
        self.tyb, self.tye = tile_row_range(rank, world, height, tile)
        self.rows_px = self.per * tile                     # pixel rows of one gathered piece (a clipped strip leaves its tail unused)
        self.piece = torch.zeros((3, self.rows_px, width), dtype=torch.float32, device=device)
        self.gathered = torch.zeros((world, 3, self.rows_px, width), dtype=torch.float32, device=device)
        self.image = torch.empty((3, height, width), dtype=torch.float32, device=device)

    def strip_rows(self) -> int:
        return max(0, min(self.H, self.tile * self.tye) - self.tile * self.tyb)

    def render(self, render_rows):
        """This rank's strip -> all-gather -> the whole image (on every rank)."""
        n = self.strip_rows()
        if n > 0:
            # the library writes [3][n][W] contiguously; the piece is [3][rows_px][W]: render into a view when they agree
            if n == self.rows_px:
                render_rows(self.tyb, self.tye, self.piece)
            else:
                tmp = self.torch.empty((3, n, self.W), dtype=self.torch.float32, device=self.piece.device)
                render_rows(self.tyb, self.tye, tmp)
                self.piece[:, :n].copy_(tmp)
        if self.dist is not None and self.dist.is_initialized() and self.world > 1:
            # (output = the pieces concatenated along dim 0, the form every backend accepts)
            self.dist.all_gather_into_tensor(self.gathered.view(self.world * 3, self.rows_px, self.W), self.piece)
        else:
            self.gathered[0].copy_(self.piece)
        # piece r holds image rows [r rows_px, (r + 1) rows_px): stack them plane by plane and drop the clipped tail
        stacked = self.gathered.permute(1, 0, 2, 3).reshape(3, self.world * self.rows_px, self.W)
        self.image.copy_(stacked[:, :self.H])
        return self.image

    def bytes_gathered_per_frame(self) -> int:
        return int(self.gathered.numel() * 4)
