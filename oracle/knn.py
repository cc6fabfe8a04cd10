"""Overlap pruning's neighbour statistic, brute force -- TEST INFRASTRUCTURE (see oracle/__init__.py).

P:167-173 (§4.3): a Gaussian is removed when "the average distance of its three nearest neighbors falls below a pre-defined
distance threshold d_OP^(l)", d_OP^(l) = s_min^(l) / 2; all removals are decided on the set as given ("removes all
Gaussians whose mean < d_OP simultaneously"; with n <= 3 Gaussians k = n - 1, with n <= 1 nothing happens).

The definition written out: all n^2 distances, the k smallest per row.  Floating point decides an integer here (remove or
keep), so the precision is fixed and the kernel takes the decision in the same one: fp32, one rounding per operation,
d^2 = (dx dx + dy dy) + dz dz, mean = ((sqrt d1 + sqrt d2) + sqrt d3) / k with d1 <= d2 <= d3, remove iff mean < 0.5f s_min.
Pins (tests/test_knn.py): the printed examples of S:266-268, scipy's k-d tree (fp64) on random sets, hand-made lattices.
"""
from __future__ import annotations

import numpy as np


def mean_knn_distance(mean, k: int = 3, block: int = 512):
    """fp32 array [n]: the average distance to the min(k, n - 1) nearest neighbours (inf for n <= 1)."""
    x = np.ascontiguousarray(mean, dtype=np.float32)
    n = x.shape[0]
    kk = min(k, n - 1)
    out = np.full(n, np.inf, np.float32)
    if kk < 1:
        return out
    for b in range(0, n, block):
        e = min(n, b + block)
        d = x[None, :, :] - x[b:e, None, :]                                     # [rows, n, 3]: other - self, fp32
        d2 = (d[..., 0] * d[..., 0] + d[..., 1] * d[..., 1]) + d[..., 2] * d[..., 2]
        d2[np.arange(e - b), np.arange(b, e)] = np.inf                          # not its own neighbour
        near = np.sort(np.partition(d2, kk - 1, axis=1)[:, :kk], axis=1)        # the kk smallest, ascending
        s = np.sqrt(near[:, 0])
        for j in range(1, kk):
            s = s + np.sqrt(near[:, j])
        out[b:e] = s / np.float32(kk)
    return out


def overlap_prune_mask(mean, s_min: float):
    """uint8 [n]: 1 = removed (mean 3-NN distance < d_OP = s_min / 2), and the distances."""
    m = mean_knn_distance(mean)
    d_op = np.float32(0.5) * np.float32(s_min)
    return (m < d_op).astype(np.uint8), m
