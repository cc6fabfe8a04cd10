"""flod_overlap_prune_static: the overlap-prune neighbour search (§4.3) for callers that cannot allocate device
memory.  Its scratch is a fixed device array inside the library instead of a caller-owned workspace; everything else is
flod_overlap_prune, so the two must agree bit for bit -- also on a second call, when the array still holds the first
call's contents.  (Named so that pytest collects it last.)"""
import numpy as np
import pytest


def _points(seed, n):
    """Clustered means with near-duplicates: both kept and removed Gaussians, decided and undecided distances."""
    rng = np.random.default_rng(seed)
    x = rng.normal(0, 0.4, (n, 3)).astype(np.float32)
    k = n // 8
    x[:k] = x[k:2 * k] + rng.normal(0, 2e-3, (k, 3)).astype(np.float32)
    return x


def _static(pkg, torch, x, s_min):
    """One call of the no-allocation entry point on preallocated outputs; returns numpy copies after a synchronise."""
    mean = torch.from_numpy(x).cuda()
    n = x.shape[0]
    remove = torch.full((n,), 7, dtype=torch.uint8, device="cuda")            # every element must be overwritten
    dist = torch.full((n,), -1.0, dtype=torch.float32, device="cuda")
    lo = x.min(axis=0) if n else np.zeros(3, np.float32)
    pkg.overlap_prune_static(mean, s_min, lo, remove, dist)
    torch.cuda.synchronize()
    return remove.cpu().numpy(), dist.cpu().numpy()


@pytest.mark.gpu
def test_static_scratch_entry_point_matches_workspace_path_on_two_calls_in_a_row():
    import torch
    from paper_2408_12894_b200 import build
    build.build()
    import paper_2408_12894_b200 as pkg
    # the second call is smaller (and differently laid out) than the first, the third is larger again: whatever the
    # array keeps from an earlier call lies inside the regions a later call uses
    for seed, n, s_min in ((1, 20000, 0.06), (2, 3001, 0.2), (3, 50000, 0.03)):
        x = _points(seed, n)
        want_rm, want_dist = pkg.overlap_prune(torch.from_numpy(x).cuda(), s_min)
        want_rm, want_dist = want_rm.cpu().numpy(), want_dist.cpu().numpy()
        got_rm, got_dist = _static(pkg, torch, x, s_min)
        assert np.array_equal(got_rm, want_rm)                                 # the removed set, exactly
        assert np.array_equal(got_dist, want_dist)                             # same kernels, same bits (+inf included)
        assert 0 < int(want_rm.sum()) < n and np.isfinite(want_dist).any()     # the case decides something
    # the same input twice in a row gives the same answer twice
    x = _points(4, 12345)
    a = _static(pkg, torch, x, 0.1)
    b = _static(pkg, torch, x, 0.1)
    assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1])


@pytest.mark.gpu
def test_static_scratch_entry_point_limits():
    import torch
    from paper_2408_12894_b200 import build
    build.build()
    import paper_2408_12894_b200 as pkg
    lib = pkg.load_library()
    assert lib.flod_overlap_prune_static_setup() == 0
    n_max = pkg.overlap_prune_static_max_n()
    assert n_max == 1 << 18
    # one point beyond the maximum is rejected with its own error code, before anything is launched
    mean = torch.zeros((n_max + 1, 3), dtype=torch.float32, device="cuda")
    remove = torch.full((n_max + 1,), 7, dtype=torch.uint8, device="cuda")
    with pytest.raises(pkg.FlodError) as e:
        pkg.overlap_prune_static(mean, 0.1, (0.0, 0.0, 0.0), remove)
    assert e.value.code == -8 and str(n_max) in str(e.value)
    torch.cuda.synchronize()
    assert int(remove.min()) == 7
    # the maximum itself is served, and agrees with the workspace path
    x = _points(5, n_max)
    want_rm, want_dist = pkg.overlap_prune(torch.from_numpy(x).cuda(), 0.02)
    got_rm, got_dist = _static(pkg, torch, x, 0.02)
    assert np.array_equal(got_rm, want_rm.cpu().numpy()) and np.array_equal(got_dist, want_dist.cpu().numpy())
    # n = 0 is a no-op; a call without distances leaves them alone
    pkg.overlap_prune_static(torch.zeros((0, 3), dtype=torch.float32, device="cuda"), 0.1, (0.0, 0.0, 0.0),
                             torch.zeros((0,), dtype=torch.uint8, device="cuda"))
    x = _points(6, 1000)
    remove = torch.zeros((1000,), dtype=torch.uint8, device="cuda")
    pkg.overlap_prune_static(torch.from_numpy(x).cuda(), 0.1, x.min(axis=0), remove, None)
    torch.cuda.synchronize()
    assert np.array_equal(remove.cpu().numpy(), pkg.overlap_prune(torch.from_numpy(x).cuda(), 0.1, with_distances=False)[0].cpu().numpy())
