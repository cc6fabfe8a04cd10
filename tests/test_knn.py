"""Overlap pruning's 3-nearest-neighbour rule (§4.3): the brute-force oracle against what the
paper / SPEC and a library routine fix (CPU), then the CUDA kernel against the oracle (GPU, through the C ABI)."""
import math

import numpy as np
import pytest

from oracle.knn import mean_knn_distance, overlap_prune_mask


# ------------------------------------------------------------------------------------ pins of the oracle (CPU)

def test_printed_examples():
    """d_OP at level 1 with tau = 0.2 is 0.1; the corners of a unit square have mean 3-NN distance
    (1 + 1 + sqrt 2)/3 = 1.138 > 0.5: none removed; two coincident Gaussians: both removed."""
    sq = np.array([[0, 0, 0], [1, 0, 0], [0, 1, 0], [1, 1, 0]], np.float32)
    mask, m = overlap_prune_mask(sq, 1.0)                       # d_OP = 0.5
    assert mask.tolist() == [0, 0, 0, 0]
    np.testing.assert_allclose(m, (2 + math.sqrt(2)) / 3, rtol=1e-6)
    mask, m = overlap_prune_mask(np.array([[0.3, 0.2, 0.1]] * 2, np.float32), 0.2)
    assert mask.tolist() == [1, 1] and m.tolist() == [0.0, 0.0]
    # the threshold is HALF the scale constraint: spacing 0.09 < 0.1 = 0.2 / 2 is removed, spacing 0.11 is kept
    line = lambda h: np.stack([np.arange(20) * h, np.zeros(20), np.zeros(20)], 1).astype(np.float32)
    assert overlap_prune_mask(line(0.06), 0.2)[0][5] == 1       # interior point: mean (h + h + 2h)/3 = 0.08
    assert overlap_prune_mask(line(0.08), 0.2)[0][5] == 0       # 0.1067 >= 0.1
    # n <= 1: nothing; n = 2, 3: k = n - 1
    assert overlap_prune_mask(np.zeros((1, 3), np.float32), 0.2)[0].tolist() == [0]
    tri = np.array([[0, 0, 0], [0.03, 0, 0], [0, 0.04, 0]], np.float32)
    np.testing.assert_allclose(mean_knn_distance(tri), [0.035, 0.04, 0.045], rtol=1e-6)


def test_simple_cubic_lattice_closed_form():
    """Interior points of a cubic lattice of spacing h: three nearest neighbours at distance h exactly."""
    h = 0.125
    g = np.stack(np.meshgrid(*[np.arange(6) * h] * 3, indexing="ij"), -1).reshape(-1, 3).astype(np.float32)
    m = mean_knn_distance(g).reshape(6, 6, 6)
    assert (m == np.float32(h)).all()                          # corners have exactly three neighbours at h as well


def test_against_a_kd_tree():
    """A library routine on the same definition: scipy's cKDTree (fp64).  The fp32 decision may differ from the fp64 one
    only where the mean sits within rounding of d_OP."""
    from scipy.spatial import cKDTree
    rng = np.random.default_rng(5)
    for n, s_min in ((500, 0.2), (3000, 0.1), (4000, 0.05)):
        x = rng.normal(0, 0.5, (n, 3)).astype(np.float32)
        x[: n // 10] = x[n // 10: 2 * (n // 10)] + rng.normal(0, 1e-3, (n // 10, 3)).astype(np.float32)   # near-duplicates
        d, _ = cKDTree(x.astype(np.float64)).query(x.astype(np.float64), k=4)
        want = d[:, 1:].mean(axis=1)
        mask, m = overlap_prune_mask(x, s_min)
        np.testing.assert_allclose(m, want, rtol=2e-5, atol=1e-6)
        clear = np.abs(want - s_min / 2) > 1e-5 * s_min
        assert np.array_equal(mask[clear], (want < s_min / 2)[clear].astype(np.uint8)) and 0 < mask.sum() < n


# ------------------------------------------------------------------------------------ the CUDA kernel (GPU)

def _gpu(x, s_min):
    import torch
    from paper_2408_12894_b200 import build
    build.build()
    import paper_2408_12894_b200 as pkg
    rm, dist = pkg.overlap_prune(torch.from_numpy(np.ascontiguousarray(x, np.float32)).cuda(), s_min)
    return rm.cpu().numpy(), dist.cpu().numpy()


def _check(x, s_min):
    mask, m = overlap_prune_mask(x, s_min)
    rm, dist = _gpu(x, s_min)
    assert np.array_equal(rm, mask)                              # the removed set: exactly the oracle's
    known = np.isfinite(dist)
    assert np.array_equal(dist[known], m[known])                 # bit for bit where the kernel decides the mean
    assert (m[~known] >= np.float32(0.5) * np.float32(s_min)).all()      # "+inf" only ever means "not below d_OP"
    # ... and it is decided whenever the third neighbour lies within 3 d_OP
    return int(mask.sum()), int(known.sum())


@pytest.mark.gpu
@pytest.mark.parametrize("seed", range(12))
def test_kernel_equals_brute_force_on_random_configurations(seed):
    """the removed set equals the O(n^2) oracle's on random configurations (clusters, near-duplicates, exact
    duplicates, isolated points, n from 0 to 5000, thresholds from far below to far above the typical spacing)."""
    rng = np.random.default_rng(1000 + seed)
    n = int(rng.integers(0, 5000)) if seed else 0
    x = rng.normal(0, 1.0, (n, 3)) * rng.uniform(0.2, 3.0, 3)
    if n > 50:
        x[: n // 5] = x[n // 5: 2 * (n // 5)] + rng.normal(0, 10 ** rng.uniform(-4, -1), (n // 5, 3))
        x[-40:] = np.tile(x[:10], (4, 1))                        # exact duplicates, five of each: mean distance 0
        x[-50:-40] += 50.0                                       # a far-away clump
    s_min = float(10 ** rng.uniform(-2.5, 0.3))
    removed, known = _check(x.astype(np.float32), s_min)
    if n > 50:
        assert removed >= 50


@pytest.mark.gpu
def test_kernel_small_sets_and_printed_examples():
    for x in (np.zeros((1, 3)), np.array([[0.3, 0.2, 0.1]] * 2), np.array([[0, 0, 0], [0.03, 0, 0], [0, 0.04, 0]]),
              np.array([[0, 0, 0], [1, 0, 0], [0, 1, 0], [1, 1, 0]], float)):
        for s_min in (0.05, 0.2, 1.0, 4.0):
            _check(x.astype(np.float32), s_min)
    import paper_2408_12894_b200 as pkg
    import torch
    with pytest.raises(pkg.FlodError):
        pkg.overlap_prune(torch.zeros((4, 3), device="cuda"), 0.0)      # the rule is for levels below L_max (s_min > 0)


@pytest.mark.gpu
def test_kernel_at_the_size_of_a_level():
    """Config 1's level 3 (600,000 Gaussians, the level's own positions, d_OP = s_min^(3) / 2 = 0.025): against scipy's
    k-d tree in fp64 away from the threshold, and against the brute-force oracle on a sample of rows."""
    from scipy.spatial import cKDTree
    import flod_synth as fs
    lv = fs.make_scene(1, levels=[3]).levels[0]
    x = lv.mean
    x64 = x.astype(np.float64)
    d, _ = cKDTree(x64).query(x64, k=4, workers=-1)
    want = d[:, 1:].mean(axis=1)
    for s_min in (lv.s_min, 8 * lv.s_min):                     # the level's own constraint (sparse scene: nothing to remove), and 8x
        rm, dist = _gpu(x, s_min)
        clear = np.abs(want - s_min / 2) > 1e-5 * s_min
        assert np.array_equal(rm[clear], (want < s_min / 2)[clear].astype(np.uint8)) and (~clear).sum() < 100
        known = np.isfinite(dist)
        np.testing.assert_allclose(dist[known], want[known], rtol=2e-5, atol=1e-6)
        assert (want[~known] >= s_min / 2).all()
        print(f"level 3 of config 1, s_min {s_min:.3f}: {int(rm.sum())} of {len(x)} removed, mean decided for {int(known.sum())}")
    assert rm.sum() > 10000
