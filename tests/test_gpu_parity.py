"""Parity of the CUDA path (through the C ABI) with the CPU oracle on the same seeded inputs.

Bit-exact: activation, selection masks, projected geometry (mu', depth, conic, rects), per-tile pair counts,
the sorted (tile, depth, gid) sequence, frame counters.  Floating point: colours to 1e-5, images to max-abs 1e-3
per channel (north_star) with the envelope rule of DESIGN §3 for the 1/255 skip.
"""
import math

import numpy as np
import pytest

import flod_synth as fs
import oracle
from helpers import camera, level
from oracle import OracleScene, SKIP_THR

pytestmark = pytest.mark.gpu

DELTA = 2.0 ** -16


@pytest.fixture(scope="module")
def pkg():
    from paper_2408_12894_b200 import build
    build.build()
    import paper_2408_12894_b200 as p
    return p


def make_renderer(pkg, levels, sh_degree, width, height, max_pairs=1 << 20, flags=None):
    r = pkg.Renderer(0)
    r.upload_levels(levels, sh_degree)
    r.set_workspace(width, height, max_pairs)
    r.set_options(pkg.FLOD_OPT_DEBUG if flags is None else flags)
    return r


def check_image(gpu, fr, tol=1e-3, brute=False):
    """north_star tolerance with the envelope rule; returns (max abs diff, number of marginal pixels).
    brute=True compares with per-pixel compositing over ALL depth-sorted Gaussians (no tiles, no rects)."""
    ref = fr.composite(brute=brute)
    d = np.abs(gpu.astype(np.float64) - ref)
    bad = d > tol
    n_marginal = 0
    if bad.any():
        lo = fr.composite(skip_thr=SKIP_THR * (1 - DELTA), brute=brute)
        hi = fr.composite(skip_thr=SKIP_THR * (1 + DELTA), brute=brute)
        mn = np.minimum(np.minimum(ref, lo), hi) - tol
        mx = np.maximum(np.maximum(ref, lo), hi) + tol
        marginal = (np.abs(lo - ref) > 1e-5) | (np.abs(hi - ref) > 1e-5)
        n_marginal = int(marginal.any(axis=0).sum())
        still = bad & ~(marginal & (gpu >= mn) & (gpu <= mx))
        assert not still.any(), f"{int(still.sum())} channel values off by more than {tol}: max {d[still].max():.3e}"
    return float(d.max()), n_marginal


def check_frame(r, osc, cam, l_start, l_end, gamma, ref_pos=None, image=True):
    """Render one frame on the GPU and compare every checked intermediate with the oracle's frame."""
    r.set_selection_reference(ref_pos)
    img = r.render(cam, l_start, l_end, gamma).cpu().numpy()
    st = r.get_stats()
    fr = osc.frame(cam, l_start, l_end, gamma, ref_pos, pair_rule=r.pair_rule)
    c = fr.counts
    assert (st["n_scan"], st["n_sel"], st["n_front"], st["n_vis"], st["n_pairs"]) == (
        c["n_scan"], c["n_sel"], c["n_front"], c["n_vis"], c["n_pairs"])
    # level-selection mask: bit-exact
    assert np.array_equal(r.debug_mask(), fr.mask)
    # per-tile pair counts: bit-exact
    assert np.array_equal(r.debug_tile_counts(fr.TX * fr.TY), fr.tile_counts)
    # projected records in ascending gid
    pr = r.debug_projected(st["n_vis"])
    vis = np.nonzero(fr.state == oracle.ST_VISIBLE)[0]
    assert np.array_equal(pr["gid"], vis.astype(np.uint32))
    assert np.array_equal(pr["mu2d"], fr.mu2d[vis]) and np.array_equal(pr["depth"], fr.depth[vis])
    assert np.array_equal(pr["conic"], fr.conic[vis]) and np.array_equal(pr["rect"], fr.rect[vis])
    assert np.array_equal(pr["opacity"], osc.opacity[vis])
    if len(vis):
        assert np.abs(pr["rgb"].astype(np.float64) - fr.rgb[vis]).max() <= 1e-5
    # the sorted (tile, depth, gid) sequence is unique, so it must be identical
    sp = r.debug_sorted_pairs(st["n_pairs"])
    tile, depth, gid = fr.sorted_pairs()
    assert np.array_equal(sp["tile"], tile) and np.array_equal(sp["depth"], depth) and np.array_equal(sp["gid"], gid)
    if image:
        return check_image(img, fr), img, fr
    return None, img, fr


# ------------------------------------------------------------------------------------ config 0

@pytest.fixture(scope="module")
def config0(pkg):
    sc = fs.make_scene(0)
    cam = fs.make_poses(0)[0]
    return sc, cam, OracleScene(sc.levels, sc.sh_degree), make_renderer(pkg, sc.levels, sc.sh_degree, cam.width, cam.height)


def test_activation_bit_exact(config0):
    """Step a0 (Eq. 1): the library's host activation equals the oracle's bit for bit."""
    sc, cam, osc, r = config0
    act = r.debug_activated()
    assert np.array_equal(act[:, :6], osc.cov)
    assert np.array_equal(act[:, 6], osc.opacity)
    dead = osc.dead.astype(bool)
    assert np.array_equal(act[~dead, 7], osc.kappa[~dead]) and (act[dead, 7] == -1.0).all()


def test_config0_max_level(config0):
    sc, cam, osc, r = config0
    (dmax, nm), img, fr = check_frame(r, osc, cam, 2, 2, 1.0)
    assert fr.counts["n_pairs"] > 10000 and dmax <= 1e-3 + 4e-3


def test_config0_both_pair_rules(pkg, config0):
    """R13 / R26: the box rule and the ellipse rule give their own per-tile counts and pair sequences --
    each exactly the oracle's for that rule -- and the same image bit for bit (a dropped tile holds no pixel with
    alpha >= 1/255, so no blended term changes)."""
    sc, cam, osc, r = config0
    imgs, pairs = {}, {}
    try:
        for rule in (pkg.PAIR_RULE_BOX, pkg.PAIR_RULE_ELLIPSE):
            r.set_pair_rule(rule)
            for (ls, le) in ((2, 2), (1, 2)):
                _, img, fr = check_frame(r, osc, cam, ls, le, 1.0)
                imgs[rule, ls] = img
                pairs[rule, ls] = fr.counts["n_pairs"]
    finally:
        r.set_pair_rule(pkg.PAIR_RULE_BOX)
    for ls in (2, 1):
        assert np.array_equal(imgs[1, ls], imgs[2, ls]) and pairs[2, ls] < 0.95 * pairs[1, ls]
    with pytest.raises(pkg.FlodError):
        r.set_pair_rule(3)


def test_config0_selective(config0):
    """BASELINE.json config 0: selective render with levels {1,2}, gamma = 1 px."""
    sc, cam, osc, r = config0
    (dmax, nm), img, fr = check_frame(r, osc, cam, 1, 2, 1.0)
    m = fr.mask
    assert 0 < m[:1000].sum() < 1000 and 0 < m[1000:].sum() < 4000
    for gamma in (0.5, 2.0, 4.0):
        check_frame(r, osc, cam, 1, 2, gamma)
    check_frame(r, osc, cam, 1, 2, 1.0, ref_pos=[0.3, -0.2, 0.1])


def test_config0_single_level_equals_selective_single_range(config0):
    """a single-level range renders bit-identically whatever gamma is."""
    sc, cam, osc, r = config0
    a = r.render(cam, 1, 1, 1.0).cpu().numpy()
    b = r.render(cam, 1, 1, 7.0).cpu().numpy()
    assert np.array_equal(a, b)
    check_frame(r, osc, cam, 1, 1, 1.0)


def test_determinism(config0):
    sc, cam, osc, r = config0
    a = r.render(cam, 1, 2, 1.0).cpu().numpy()
    for _ in range(3):
        assert np.array_equal(a, r.render(cam, 1, 2, 1.0).cpu().numpy())


def test_brute_force_parity_on_tiny_input(config0):
    """north_star: GPU image against per-pixel compositing over ALL depth-sorted Gaussians (no tiles)."""
    sc, cam, osc, r = config0
    for (ls, le) in ((1, 2), (2, 2)):
        img = r.render(cam, ls, le, 1.0).cpu().numpy()
        check_image(img, osc.frame(cam, ls, le, 1.0, pair_rule=r.pair_rule), brute=True)


# ------------------------------------------------------------------------- edge cases, small scenes

def _rand_levels(rng, counts, s_min, extent=1.5, sh_degree=0, zrange=(0.3, 6.0), logs=(-4.0, -1.0)):
    out = []
    K = (sh_degree + 1) ** 2
    for i, n in enumerate(counts):
        pos = np.stack([rng.uniform(-extent, extent, n), rng.uniform(-extent, extent, n), rng.uniform(*zrange, n)], axis=1)
        sh = rng.normal(0, 0.25, (n, K, 3)); sh[:, 0, :] += 0.8
        lv = level(i + 1, s_min[i], pos.reshape(n, 3), np.exp(rng.uniform(*logs, (n, 3))), quat=rng.normal(size=(n, 4)) + 1e-3,
                   logit=rng.normal(0, 2.0, n), sh=sh)
        if n == 0:
            lv.quat = np.zeros((0, 4), np.float32)
        out.append(lv)
    return out


@pytest.mark.parametrize("seed,counts,wh,deg", [
    (1, (300, 700), (100, 60), 0),          # ragged image (not a multiple of 16)
    (2, (1, 1), (16, 16), 1),               # one tile, one Gaussian per level
    (3, (0, 513), (33, 17), 2),             # empty level, ragged everything
    (4, (257, 0), (64, 48), 3),             # empty top level, block-boundary count
    (5, (5000, 9000, 14000), (250, 130), 3),  # several preprocess blocks / sort tiles, degree 3
    (6, (255, 256, 257), (17, 200), 0),
])
def test_random_scenes(pkg, seed, counts, wh, deg):
    rng = np.random.default_rng(seed)
    s_min = np.sort(np.exp(rng.uniform(-4, -1, len(counts))))[::-1].copy()
    s_min[-1] = 0.0
    lv = _rand_levels(rng, counts, s_min, sh_degree=deg)
    cam = camera(width=wh[0], height=wh[1], f=float(rng.uniform(40, 120)), bg=tuple(rng.uniform(0, 1, 3)))
    osc = OracleScene(lv, deg)
    r = make_renderer(pkg, lv, deg, wh[0], wh[1], max_pairs=1 << 21)
    L = len(counts)
    for rule in (pkg.PAIR_RULE_ELLIPSE, pkg.PAIR_RULE_BOX):
        r.set_pair_rule(rule)
        check_frame(r, osc, cam, L, L, 1.0)
        check_frame(r, osc, cam, 1, L, 2.0)
        check_frame(r, osc, cam, 1, 1, 1.0)
    r.close()


def test_tile_counts_of_rects_across_tile_group_boundaries(pkg):
    """Step a5: k_geometry counts the tiles of a rect of at most 2x2 groups of 2x2 tiles in per-group float4 counters
    and those of a larger rect in the 2-D difference grid (DESIGN 6.1); the tile scan sums the two.  Isotropic Gaussians
    of graded sizes at controlled screen positions produce every combination of rect origin parity and rect extent
    1..6 tiles in x and y, on an image whose tile grid is odd in both directions (a group column / row hangs over the
    edge).  Per-tile counts, the sorted sequence and the image against the oracle, both pair rules, and a strip."""
    f, z, W, H = 100.0, 10.0, 201, 171                       # 13 x 11 tiles
    means, scales = [], []
    for ext in (0.02, 0.35, 0.8, 1.3, 1.9, 2.6):             # alpha = 1/255 radius from about 1 to about 45 pixels
        for ty in range(0, 11, 1):
            for tx in range(0, 13, 1):
                # a centre near a tile corner, near a tile centre, near a group corner -- per size another offset
                ox, oy = [(1.0, 1.0), (8.0, 8.0), (15.0, 3.0), (4.0, 15.5), (0.2, 9.0), (12.0, 0.3)][int(ext * 10) % 6]
                u, v = 16.0 * tx + ox, 16.0 * ty + oy
                means.append(((u - W / 2.0) * z / f, (v - H / 2.0) * z / f, z + 0.001 * len(means)))
                scales.append(ext)
    means, scales = np.array(means), np.array(scales)[:, None] * np.ones(3)
    rng = np.random.default_rng(5)
    lv = [level(1, 0.0, means, scales, opacity=rng.uniform(0.05, 0.95, len(means)), rgb=rng.uniform(0, 1, (len(means), 3)))]
    cam = camera(width=W, height=H, f=f, bg=(0.1, 0.2, 0.3))
    osc = OracleScene(lv, 0)
    r = make_renderer(pkg, lv, 0, W, H, max_pairs=1 << 21)
    for rule in (pkg.PAIR_RULE_BOX, pkg.PAIR_RULE_ELLIPSE):
        r.set_pair_rule(rule)
        (dmax, nm), img, fr = check_frame(r, osc, cam, 1, 1, 1.0)
        rc = fr.rect[fr.state == oracle.ST_VISIBLE].astype(np.int64)
        gw, gh = (rc[:, 2] + 1) // 2 - rc[:, 0] // 2, (rc[:, 3] + 1) // 2 - rc[:, 1] // 2
        small = (gw <= 2) & (gh <= 2)
        assert small.sum() > 200 and (~small).sum() > 200            # both counting paths are exercised
        shapes = {(int(a[0]) & 1, int(a[1]) & 1, int(a[2] - a[0]), int(a[3] - a[1])) for a in rc}
        assert len(shapes) > 60                                      # origin parities x extents
    r.set_pair_rule(pkg.PAIR_RULE_BOX)
    full = r.render(cam, 1, 1, 1.0).cpu().numpy()
    img, _ = _assemble_strips(r, cam, 1, 1, 1.0, 3)                  # strips that begin on odd tile rows
    assert np.array_equal(img, full)
    r.close()


def test_screen_filling_rects_shared_counter_duplication(pkg):
    """Step a6 on frames of VERY large rects (mean above 1024 tiles per Gaussian): k_duplicate_shared by default, without
    the test knob.  300 Gaussians that each cover most of a 592 x 560 image (37 x 35 = 1295 tiles) plus a few small
    ones; counts, sorted sequence and image against the oracle under both pair rules."""
    rng = np.random.default_rng(77)
    W, H, f, z = 592, 560, 120.0, 6.0
    n_big, n_small = 300, 40
    mean = np.concatenate([np.c_[rng.uniform(-2, 2, n_big), rng.uniform(-2, 2, n_big), z + rng.uniform(0, 3, n_big)],
                           np.c_[rng.uniform(-10, 10, n_small), rng.uniform(-10, 10, n_small), z + rng.uniform(0, 3, n_small)]])
    scale = np.concatenate([np.exp(rng.uniform(2.0, 2.6, (n_big, 3))), np.exp(rng.uniform(-3, -2, (n_small, 3)))])
    q = rng.normal(size=(n_big + n_small, 4)); q /= np.linalg.norm(q, axis=1, keepdims=True)
    lv = [level(1, 0.0, mean, scale, quat=q, opacity=rng.uniform(0.02, 0.3, n_big + n_small), rgb=rng.uniform(0, 1, (n_big + n_small, 3)))]
    cam = camera(width=W, height=H, f=f, bg=(0.2, 0.1, 0.0))
    osc = OracleScene(lv, 0)
    r = make_renderer(pkg, lv, 0, W, H, max_pairs=1 << 20)
    for rule in (pkg.PAIR_RULE_BOX, pkg.PAIR_RULE_ELLIPSE):
        r.set_pair_rule(rule)
        (dmax, nm), img, fr = check_frame(r, osc, cam, 1, 1, 1.0)
        if rule == pkg.PAIR_RULE_BOX:
            assert fr.counts["n_pairs"] > 1024 * fr.counts["n_vis"]        # the default threshold of the shared-counter kernel
        check_frame(r, osc, cam, 1, 1, 1.0)                                # (a second frame: after the hint reached the host)
    r.close()


def test_empty_scene_and_all_culled(pkg):
    """nothing to draw -> background; also everything behind the camera / dead."""
    lv = level(1, 0.0, np.zeros((0, 3)), 0.1)
    lv.quat = np.zeros((0, 4), np.float32)
    cam = camera(width=40, height=24, bg=(0.25, 0.5, 0.75))
    r = make_renderer(pkg, [lv], 0, 40, 24)
    img = r.render(cam, 1, 1, 1.0).cpu().numpy()
    assert (img[0] == 0.25).all() and (img[1] == 0.5).all() and (img[2] == 0.75).all()
    st = r.get_stats()
    assert st["n_pairs"] == 0 and st["n_vis"] == 0 and st["n_scan"] == 0
    r.close()
    lv = level(1, 0.0, [[0, 0, -1.0], [0, 0, 0.1], [0, 0, 2.0]], 0.1, logit=[0.0, 0.0, -9.0])
    r = make_renderer(pkg, [lv], 0, 40, 24)
    osc = OracleScene([lv], 0)
    (dmax, _), img, fr = check_frame(r, osc, cam, 1, 1, 1.0)
    assert fr.counts["n_vis"] == 0 and (img[1] == 0.5).all()
    r.close()


def test_screen_filling_and_degenerate_gaussians(pkg):
    """Maximum footprints (every tile), a Gaussian beside the frustum (Jacobian clamp R8), exact depth ties."""
    cam = camera(width=96, height=64, f=80.0)
    pos = [[0, 0, 1.0], [0.05, 0.02, 1.0], [6.0, 0.1, 1.0], [0, 0, 1.0], [-0.3, 0.2, 0.5], [0.0, 0.0, 0.2000001]]
    sc = [[3.0, 3.0, 3.0], [0.5, 0.001, 0.001], [0.4, 0.4, 0.4], [0.02, 0.02, 0.02], [1.0, 0.0005, 0.3], [0.01, 0.01, 0.01]]
    lv = level(1, 0.0, pos, np.array(sc), quat=[[1, 0, 0, 0], [0.9, 0.1, 0.3, 0.2], [1, 0, 0, 0], [1, 0, 0, 0], [0.3, 0.5, 0.1, 0.8], [1, 0, 0, 0]],
               opacity=[0.3, 0.9, 0.8, 0.99, 0.6, 0.5], rgb=[[1, 0, 0], [0, 1, 0], [0, 0, 1], [1, 1, 0], [0, 1, 1], [1, 0, 1]])
    r = make_renderer(pkg, [lv], 0, 96, 64)
    osc = OracleScene([lv], 0)
    for rule in (pkg.PAIR_RULE_BOX, pkg.PAIR_RULE_ELLIPSE):
        r.set_pair_rule(rule)
        (dmax, _), img, fr = check_frame(r, osc, cam, 1, 1, 1.0)
        assert fr.n_tiles.max() == fr.TX * fr.TY
    r.close()


def test_sort_corner_cases_long_lists_and_depth_plateaus(pkg):
    """Per-tile ordering (R15) where the per-tile sort leaves its common path: tile lists far longer than its
    shared-memory capacity, thousands of exactly equal depths in one tile (planes facing the camera: the order is
    decided by gid alone), and nested clusters of nearly equal depths inside a wide depth range."""
    rng = np.random.default_rng(77)
    n_plane, n_cl, n_far = 10000, 3000, 2000
    # two planes of identical camera depth (identity pose: depth = z exactly), small footprints over 2x2 tiles
    xy = rng.uniform(-0.06, 0.06, (2 * n_plane, 2))
    z = np.repeat([2.0, 2.5], n_plane)
    plane = np.column_stack([xy * z[:, None], z])
    # nested clusters: depths 4 + k * 2^-20 (adjacent fp32 values around 4), and a wide-range background
    cl = np.column_stack([rng.uniform(-0.3, 0.3, (n_cl, 2)), 4.0 + rng.integers(0, 40, n_cl) * 2.0 ** -20])
    far = np.column_stack([rng.uniform(-2, 2, (n_far, 2)), rng.uniform(0.3, 400.0, n_far)])
    pos = np.concatenate([plane, cl, far])
    pos = pos[rng.permutation(len(pos))]
    lv = level(1, 0.0, pos, 0.004 * pos[:, 2:3] * np.ones((1, 3)), opacity=rng.uniform(0.02, 0.2, len(pos)),
               rgb=rng.uniform(0, 1, (len(pos), 3)))
    cam = camera(width=64, height=48, f=100.0)
    r = make_renderer(pkg, [lv], 0, 64, 48, max_pairs=1 << 20)
    osc = OracleScene([lv], 0)
    _, img_dbg, fr = check_frame(r, osc, cam, 1, 1, 1.0)
    assert fr.tile_counts.max() > 2 * 4096          # beyond the shared-memory path of the sort
    # blend-driven ordering (the default without a debug view): long lists are ordered only as far as the blend reads
    # them, in one or two rounds -- the image is the fully sorted frame's, bit for bit
    for flags in (0, pkg.FLOD_OPT_FULL_SORT, pkg.FLOD_OPT_PROFILE):
        r.set_options(flags)
        assert np.array_equal(r.render(cam, 1, 1, 1.0).cpu().numpy(), img_dbg)
    r.close()


def test_blend_driven_ordering_two_rounds(pkg):
    """Lists of six thousand faint Gaussians: the sorted prefix of the first round (the nearest slices, >= 1024 keys) is
    not enough for most tiles, so the second round (k_tile_sort_rest, k_blend resuming from the saved pixel state) runs;
    other tiles (opaque foreground) finish in the first.  Bit-identical to the fully sorted frame."""
    rng = np.random.default_rng(88)
    n_faint, n_front = 60000, 300
    pos = np.column_stack([rng.uniform(-1.2, 1.2, (n_faint, 2)), rng.uniform(1.0, 40.0, n_faint)])
    pos[:, :2] *= pos[:, 2:3] * 0.5
    front = np.column_stack([rng.uniform(-0.25, 0.0, (n_front, 2)), rng.uniform(0.5, 0.9, n_front)])      # covers the upper-left tiles only
    allpos = np.concatenate([pos, front])
    scale = np.concatenate([0.03 * pos[:, 2:3] * np.ones((1, 3)), 0.05 * np.ones((n_front, 3))])
    opac = np.concatenate([rng.uniform(0.01, 0.03, n_faint), np.full(n_front, 0.95)])
    lv = level(1, 0.0, allpos, scale, opacity=opac, rgb=rng.uniform(0, 1, (len(allpos), 3)))
    cam = camera(width=96, height=64, f=60.0, bg=(0.1, 0.1, 0.1))
    r = make_renderer(pkg, [lv], 0, 96, 64, max_pairs=1 << 22)
    osc = OracleScene([lv], 0)
    (dmax, _), img_dbg, fr = check_frame(r, osc, cam, 1, 1, 1.0)
    assert np.median(fr.tile_counts) > 4096 + 1024
    _, E, B, T = fr.composite(stats=True)
    assert (T > 1e-4).mean() > 0.3 and (T < 1e-4).mean() > 0.02      # both kinds of tiles exist
    r.set_options(0)
    for _ in range(2):
        assert np.array_equal(r.render(cam, 1, 1, 1.0).cpu().numpy(), img_dbg)
    # ... and strips of such a frame
    assert np.array_equal(r.render_rows(cam, 1, 1, 1.0, 1, 3).cpu().numpy(), img_dbg[:, 16:48])
    r.close()


def test_needle_gaussians_stay_within_tolerance(pkg):
    """DESIGN R25: long thin footprints (short axis at the dilation floor) are where the textbook exponent loses
    precision in fp32; the factorised form keeps the image within 1e-3."""
    rng = np.random.default_rng(12)
    n = 400
    pos = np.stack([rng.uniform(-2, 2, n), rng.uniform(-1.5, 1.5, n), rng.uniform(3.0, 8.0, n)], axis=1)
    scale = np.stack([np.exp(rng.uniform(-1.0, 1.0, n)), np.full(n, 1e-4), np.full(n, 1e-4)], axis=1)
    lv = level(1, 0.0, pos, scale, quat=rng.normal(size=(n, 4)), opacity=rng.uniform(0.3, 0.95, n), rgb=rng.uniform(0, 1, (n, 3)))
    cam = camera(width=640, height=400, f=600.0)
    r = make_renderer(pkg, [lv], 0, 640, 400)
    osc = OracleScene([lv], 0)
    r.set_pair_rule(pkg.PAIR_RULE_ELLIPSE)
    (dmax, nm), img, fr = check_frame(r, osc, cam, 1, 1, 1.0)
    r.set_pair_rule(pkg.PAIR_RULE_BOX)
    _, img1, fr1 = check_frame(r, osc, cam, 1, 1, 1.0)
    # (thin diagonal needles keep the box rule -- their determinant cancels in fp32, R26 -- the others are cut down)
    assert np.array_equal(img, img1) and fr.counts["n_pairs"] <= fr1.counts["n_pairs"]
    r.close()


def test_anisotropic_camera_off_centre_principal_point(pkg):
    """R4 and every fy / cy / lim_y term (O2-O4, Eq. 7): fx != fy, cx != W/2, cy != H/2.  With fx == fy and a centred
    principal point a swap of the two would go unnoticed on both sides."""
    rng = np.random.default_rng(61)
    lv = _rand_levels(rng, (1500, 3000, 6000), (0.08, 0.02, 0.0), extent=2.5, sh_degree=2)
    osc = OracleScene(lv, 2)
    r = make_renderer(pkg, lv, 2, 208, 136, max_pairs=1 << 22)
    for (fx, fy, cx, cy) in ((190.0, 127.0, 81.25, 90.5), (95.0, 240.0, 150.0, 20.0)):
        cam = camera(width=208, height=136, f=fx, fy=fy, cx=cx, cy=cy, bg=(0.2, 0.1, 0.3))
        check_frame(r, osc, cam, 3, 3, 1.0)
        _, _, fr = check_frame(r, osc, cam, 1, 3, fx / 47.5)       # Eq. 7 scales with fx (R4): the same bands for both cameras
        per_level = [int(fr.mask[a:b].sum()) for a, b in ((0, 1500), (1500, 4500), (4500, 10500))]
        assert per_level == [769, 1529, 40]                      # (would differ if fy were taken for f)
        check_frame(r, osc, cam, 2, 3, 0.7, ref_pos=[0.4, -0.3, 0.2])
    r.close()


def test_non_orthonormal_camera_rotation_is_rejected(pkg):
    """R is a rotation.  The covariance-free off-screen bound of k_geometry assumes it; a scaled or sheared R
    is an argument error, not a silently different image."""
    lv = level(1, 0.0, [[0, 0, 1.0]], 0.1)
    r = make_renderer(pkg, [lv], 0, 64, 64)
    for R in (np.eye(3) * 1.01, np.array([[1, 0.01, 0], [0, 1, 0], [0, 0, 1.0]])):
        with pytest.raises(pkg.FlodError) as e:
            r.render(camera(width=64, height=64, R=R), 1, 1, 1.0)
        assert e.value.code == -1
    r.render(camera(width=64, height=64), 1, 1, 1.0)
    r.close()


def test_two_contexts_in_one_process_are_independent(pkg):
    """include/flod.h: "contexts are independent".  Two contexts with different scenes and workspaces, frames
    interleaved; the per-device kernel attributes (shared-memory opt-ins) are set by every flod_create."""
    rng = np.random.default_rng(5)
    lva = _rand_levels(rng, (2000, 5000), (0.05, 0.0))
    lvb = _rand_levels(rng, (700,), (0.0,), sh_degree=1)
    cam = camera(width=96, height=80, f=90.0)
    ra = make_renderer(pkg, lva, 0, 96, 80)
    rb = make_renderer(pkg, lvb, 1, 96, 80)
    osa, osb = OracleScene(lva, 0), OracleScene(lvb, 1)
    a0 = ra.render(cam, 1, 2, 1.0).cpu().numpy()
    b0 = rb.render(cam, 1, 1, 1.0).cpu().numpy()
    for _ in range(2):
        check_frame(ra, osa, cam, 1, 2, 1.0)
        check_frame(rb, osb, cam, 1, 1, 1.0)
    assert np.array_equal(a0, ra.render(cam, 1, 2, 1.0).cpu().numpy())
    assert np.array_equal(b0, rb.render(cam, 1, 1, 1.0).cpu().numpy())
    ra.close(); rb.close()


def test_paper_rho4_ladder(pkg):
    """R7: the paper's tau = 0.2, rho = 4 ladder through Eq. 7, selective {1..5}."""
    rng = np.random.default_rng(40)
    s_min = [oracle.scale_constraint(l, 0.2, 4.0, 5) for l in range(1, 6)]
    counts = (200, 400, 800, 1600, 3200)
    lv = _rand_levels(rng, counts, s_min, extent=20.0, zrange=(0.5, 120.0), logs=(-3.0, 0.0))
    cam = camera(width=200, height=120, f=170.0)
    osc = OracleScene(lv, 0)
    r = make_renderer(pkg, lv, 0, 200, 120, max_pairs=1 << 22)
    for rng_l in ((1, 5), (3, 5), (2, 4)):
        for gamma in (0.5, 1.0, 4.0):
            _, _, fr = check_frame(r, osc, cam, rng_l[0], rng_l[1], gamma)
    r.close()


def test_errors_and_capacity(pkg):
    """Error conventions of include/flod.h: level range, gamma, workspace too small for the camera, capacity."""
    rng = np.random.default_rng(9)
    lv = _rand_levels(rng, (500, 1500), (0.05, 0.0))
    cam = camera(width=64, height=64, f=60.0)
    r = make_renderer(pkg, lv, 0, 64, 64, max_pairs=256)
    for args in ((0, 1, 1.0), (1, 3, 1.0), (2, 1, 1.0)):
        with pytest.raises(pkg.FlodError) as e:
            r.render(cam, *args)
        assert e.value.code == -2
    for gamma in (0.0, -1.0, float("nan"), float("inf")):
        with pytest.raises(pkg.FlodError) as e:
            r.render(cam, 1, 2, gamma)
        assert e.value.code == -1
    with pytest.raises(pkg.FlodError):
        r.render(camera(width=65, height=64), 1, 2, 1.0)
    # capacity: the frame needs more than 256 pairs -> flagged, required count reported, nothing out of bounds
    r.render(cam, 2, 2, 1.0)
    with pytest.raises(pkg.FlodError) as e:
        r.get_stats()
    assert e.value.code == -5
    st = r.get_stats(raise_on_overflow=False)
    need = OracleScene(lv, 0).frame(cam, 2, 2, 1.0, pair_rule=r.pair_rule).counts["n_pairs"]
    assert st["overflow"] == 1 and st["n_pairs"] == need > 256
    # the host-buffer calls block on the frame anyway, so they report the overflow themselves
    with pytest.raises(pkg.FlodError) as e:
        r.render_to_host(cam, 2, 2, 1.0)
    assert e.value.code == -5
    import torch
    side = torch.cuda.Stream(device=r.device)
    buf = torch.zeros((3, 64, 64), dtype=torch.float32).pin_memory()
    r.render_to_host_async(cam, 2, 2, 1.0, buf, side)
    with pytest.raises(pkg.FlodError) as e:
        r.wait_host()
    assert e.value.code == -5
    r.wait_host()                            # the flag was consumed: nothing pending any more
    r.set_workspace(64, 64, need)            # grow to exactly what was reported and re-render
    r.set_options(pkg.FLOD_OPT_DEBUG)
    check_frame(r, OracleScene(lv, 0), cam, 2, 2, 1.0)
    assert np.array_equal(r.render_to_host(cam, 2, 2, 1.0).numpy(), r.render(cam, 2, 2, 1.0).cpu().numpy())
    r.close()


def test_upload_validation(pkg):
    r = pkg.Renderer(0)
    ok = level(1, 0.1, [[0, 0, 1.0]], 0.1)
    bad_order = [level(2, 0.1, [[0, 0, 1.0]], 0.1), level(1, 0.0, [[0, 0, 1.0]], 0.1)]
    bad_smin = [level(1, 0.1, [[0, 0, 1.0]], 0.1), level(2, 0.2, [[0, 0, 1.0]], 0.1)]
    nan = level(1, 0.0, [[0, float("nan"), 1.0]], 0.1)
    zq = level(1, 0.0, [[0, 0, 1.0]], 0.1, quat=[[0, 0, 0, 0]])
    for lv in (bad_order, bad_smin, [nan], [zq]):
        with pytest.raises(pkg.FlodError):
            r.upload_levels(lv, 0)
    with pytest.raises(pkg.FlodError):
        r.render(camera(), 1, 1, 1.0)
    r.upload_levels([ok], 0)
    with pytest.raises(pkg.FlodError) as e:
        r.render(camera(), 1, 1, 1.0)
    assert e.value.code == -7
    r.close()


def test_levels_need_not_start_at_one(pkg):
    """R23 / P:326-327: a small device may hold only some levels; ids are what the mode refers to."""
    rng = np.random.default_rng(17)
    lv = _rand_levels(rng, (300, 600, 900), (0.1, 0.03, 0.01))
    for i, l in enumerate(lv):
        l.level = i + 2                       # levels 2,3,4 of a 5-level ladder; the top uploaded s_min is not 0
    cam = camera(width=80, height=48, f=70.0)
    osc = OracleScene(lv, 0)
    r = make_renderer(pkg, lv, 0, 80, 48)
    check_frame(r, osc, cam, 2, 4, 1.5)
    check_frame(r, osc, cam, 3, 4, 1.5)
    with pytest.raises(pkg.FlodError):
        r.render(cam, 1, 4, 1.0)
    r.close()


def test_render_to_host_matches_render(config0):
    sc, cam, osc, r = config0
    a = r.render(cam, 1, 2, 1.0).cpu().numpy()
    b = r.render_to_host(cam, 1, 2, 1.0).numpy()
    assert np.array_equal(a, b)


def test_pipelined_render_to_host_keeps_every_frame(config0):
    """flod_render_to_host_async: six frames with alternating level modes, kernels and copies on two streams, two
    images in the workspace -- every host buffer must hold exactly its own frame."""
    import torch
    sc, cam, osc, r = config0
    modes = [(2, 2), (1, 2), (1, 1), (2, 2), (1, 2), (1, 1)]
    want = [r.render(cam, ls, le, 1.0).cpu().numpy() for (ls, le) in modes]
    copy_stream = torch.cuda.Stream(device=r.device)
    bufs = [torch.zeros((3, cam.height, cam.width), dtype=torch.float32).pin_memory() for _ in modes]
    for (ls, le), b in zip(modes, bufs):
        r.render_to_host_async(cam, ls, le, 1.0, b, copy_stream)
    r.wait_host()
    for w, b in zip(want, bufs):
        assert np.array_equal(w, b.numpy())
    assert not np.array_equal(want[0], want[2])


def test_instrumented_counts_match_oracle(pkg, config0):
    """E and B of the blend stage (used for the FP32 roofline) against the oracle's per-pixel counts."""
    sc, cam, osc, _ = config0
    r = make_renderer(pkg, sc.levels, sc.sh_degree, cam.width, cam.height, flags=pkg.FLOD_OPT_COUNT | pkg.FLOD_OPT_PROFILE)
    r.render(cam, 2, 2, 1.0)
    st = r.get_stats()
    _, E, B, _ = osc.frame(cam, 2, 2, 1.0, pair_rule=r.pair_rule).composite(stats=True)
    assert abs(st["blends"] - int(B.sum())) <= max(20, 1e-3 * B.sum())
    assert abs(st["evals"] - int(E.sum())) <= max(20, 1e-3 * E.sum())
    assert st["ms_total"] > 0 and all(m >= 0 for m in st["ms_stage"])
    r.close()


# ------------------------------------------------------------------------------------ materialised G_sel

def test_subset_small_scenes_errors_and_empty_selection(pkg):
    """flod_subset_* on small inputs: three levels with the paper's rho = 4 ladder, reference positions on and off the
    camera; the error conventions; a snapshot that selects nothing renders the background."""
    rng = np.random.default_rng(21)
    lv = _rand_levels(rng, (300, 700, 2100), (0.2, 0.05, 0.0))
    osc = OracleScene(lv, 0)
    cam = camera(width=80, height=48, f=70.0, bg=(0.1, 0.2, 0.3))
    r = make_renderer(pkg, lv, 0, 80, 48)
    with pytest.raises(pkg.FlodError) as e:                      # no arena yet
        r.subset_build((0.0, 0.0, 0.0), cam.fx, 1.0)
    assert e.value.code == -7
    with pytest.raises(pkg.FlodError) as e:
        r.subset_set_arena(2, 4)
    assert e.value.code == -2
    r.subset_set_arena(1, 3)
    with pytest.raises(pkg.FlodError) as e:                      # nothing built yet
        r.render_subset(cam)
    assert e.value.code == -1
    with pytest.raises(pkg.FlodError) as e:
        r.subset_swap()
    assert e.value.code == -1
    for bad in ((float("nan"), 0.0, 0.0, cam.fx, 1.0), (0.0, 0.0, 0.0, 0.0, 1.0), (0.0, 0.0, 0.0, cam.fx, -2.0)):
        with pytest.raises(pkg.FlodError) as e:
            r.subset_build(bad[:3], bad[3], bad[4])
        assert e.value.code == -1
    for ref, gamma in (((0.0, 0.0, 0.0), 1.0), ((0.3, -0.2, 1.0), 2.0), ((5.0, 5.0, -20.0), 0.5)):
        r.subset_build(ref, cam.fx, gamma)
        with pytest.raises(pkg.FlodError) as e:                  # one rebuild at a time
            r.subset_build(ref, cam.fx, gamma)
        assert e.value.code == -1
        n_sel = r.subset_swap()
        img = r.render_subset(cam).cpu().numpy()
        st = r.get_stats()
        fr = osc.frame(cam, 1, 3, gamma, ref_pos=ref, pair_rule=r.pair_rule)
        c = fr.counts
        assert n_sel == c["n_sel"] and (st["n_front"], st["n_vis"], st["n_pairs"]) == (c["n_front"], c["n_vis"], c["n_pairs"])
        assert np.array_equal(r.debug_mask(), fr.mask)
        assert np.array_equal(r.debug_tile_counts(fr.TX * fr.TY), fr.tile_counts)
        pr = r.debug_projected(st["n_vis"])
        vis = np.nonzero(fr.state == oracle.ST_VISIBLE)[0]
        assert np.array_equal(pr["gid"], vis.astype(np.uint32)) and np.array_equal(pr["rect"], fr.rect[vis])
        check_image(img, fr)
    r.close()
    # an empty coarse level and a reference far from everything: the fine level's band [0, d) holds nothing
    lv2 = _rand_levels(rng, (0, 400), (0.05, 0.0))
    r = make_renderer(pkg, lv2, 0, 80, 48)
    r.subset_set_arena(1, 2)
    r.subset_build((0.0, 0.0, -1000.0), cam.fx, 1.0)
    assert r.subset_swap() == 0
    img = r.render_subset(cam).cpu().numpy()
    assert r.get_stats()["n_pairs"] == 0
    assert np.array_equal(img, np.broadcast_to(np.float32(cam.bg)[:, None, None], img.shape))
    r.close()


@pytest.mark.parametrize("seed", [100, 102, 105, 108, 111, 114, 120, 132])
def test_random_scenes_every_kernel_path(pkg, seed):
    """Random level counts, SH degrees, image sizes and footprints (every third seed: large footprints, mean rect area
    up to hundreds of tiles; every fourth: FLOD_OPT_SMALL_WINDOWS -> k_duplicate_shared and its tile windows from a mean
    rect of 128 tiles; seeds 108, 120, 132 are both), every checked intermediate and the
    image on the fused path, then the materialised-subset path at a random reference: bit-identical to the fused
    predicate and within tolerance of the oracle."""
    rng = np.random.default_rng(seed)
    L = int(rng.integers(1, 4)); deg = int(rng.integers(0, 4))
    counts = tuple(int(x) for x in rng.integers(0, 6000, L))
    s_min = np.sort(np.exp(rng.uniform(-4, -1, L)))[::-1].copy(); s_min[-1] = 0.0
    lv = _rand_levels(rng, counts, s_min, sh_degree=deg, logs=((-1.5, 0.5) if seed % 3 == 0 else (-4.0, -1.0)))
    W, H = int(rng.integers(16, 400)), int(rng.integers(16, 300))
    cam = camera(width=W, height=H, f=float(rng.uniform(40, 300)), bg=tuple(rng.uniform(0, 1, 3)))
    osc = OracleScene(lv, deg)
    r = make_renderer(pkg, lv, deg, W, H, max_pairs=1 << 23)
    if seed % 4 == 0:
        r.set_options(pkg.FLOD_OPT_DEBUG | pkg.FLOD_OPT_SMALL_WINDOWS)
    r.set_pair_rule(pkg.PAIR_RULE_BOX if seed % 5 == 0 else pkg.PAIR_RULE_ELLIPSE)
    check_frame(r, osc, cam, L, L, 1.0)
    check_frame(r, osc, cam, 1, L, float(rng.uniform(0.5, 4)))
    ref = rng.uniform(-2, 2, 3).astype(np.float32); gamma = float(rng.uniform(0.5, 4))
    r.subset_set_arena(1, L); r.subset_build(ref, cam.fx, gamma); r.subset_swap()
    a = r.render_subset(cam).cpu().numpy()
    r.set_selection_reference(ref)
    b = r.render(cam, 1, L, gamma).cpu().numpy()
    r.set_selection_reference(None)
    assert np.array_equal(a, b)
    check_image(a, osc.frame(cam, 1, L, gamma, ref_pos=ref, pair_rule=r.pair_rule))
    r.close()


# ------------------------------------------------------------------------------------ tile-row strips

def _assemble_strips(r, cam, ls, le, gamma, world):
    """What `world` ranks would produce (paper_2408_12894_b200.shard.RowShardedFrame without a process group: the strips
    are rendered one after the other on this GPU and stacked the way the all-gather stacks them)."""
    import torch
    from paper_2408_12894_b200.shard import RowShardedFrame
    frames = [RowShardedFrame(cam.width, cam.height, rank, world, r.device) for rank in range(world)]
    pairs = 0
    for fr in frames:
        n = fr.strip_rows()
        if n:
            fr.piece[:, :n].copy_(r.render_rows(cam, ls, le, gamma, fr.tyb, fr.tye))
            pairs += r.get_stats()["n_pairs"]
    gathered = torch.stack([fr.piece for fr in frames])
    img = gathered.permute(1, 0, 2, 3).reshape(3, world * frames[0].rows_px, cam.width)[:, :cam.height]
    return img.cpu().numpy(), pairs


@pytest.mark.parametrize("rule", [1, 2])
def test_tile_row_strips_stack_to_the_full_frame_bit_for_bit(pkg, config0, rule):
    """flod_render_rows: the strips of 2, 3 and 5 ranks, stacked, are the image flod_render writes, bit for bit, and
    together they hold exactly the frame's pairs (a rect is clipped to the strip, never listed twice)."""
    sc, cam, osc, r = config0
    r.set_pair_rule(rule)
    try:
        for (ls, le) in ((2, 2), (1, 2)):
            full = r.render(cam, ls, le, 1.0).cpu().numpy()
            n_pairs = r.get_stats()["n_pairs"]
            for world in (2, 3, 5):
                img, pairs = _assemble_strips(r, cam, ls, le, 1.0, world)
                assert np.array_equal(img, full) and pairs == n_pairs
        # a strip against the oracle directly: the oracle's frame of a camera cropped to those rows is the same strip
        strip = r.render_rows(cam, 1, 2, 1.0, 2, 5).cpu().numpy()
        assert np.array_equal(strip, full[:, 32:80])
        with pytest.raises(pkg.FlodError):
            r.render_rows(cam, 1, 2, 1.0, 3, 9)              # 128 px = 8 tile rows
        assert r.render_rows(cam, 1, 2, 1.0, 4, 4).shape == (3, 0, cam.width)
    finally:
        r.set_pair_rule(pkg.PAIR_RULE_BOX)


def test_tile_row_strips_on_a_ragged_image_with_large_footprints(pkg):
    rng = np.random.default_rng(303)
    lv = _rand_levels(rng, (3000, 5000), (0.05, 0.0), sh_degree=1, logs=(-2.5, 0.0))
    cam = camera(width=211, height=157, f=140.0, bg=(0.3, 0.2, 0.1))
    r = make_renderer(pkg, lv, 1, 211, 157, max_pairs=1 << 23)
    full = r.render(cam, 1, 2, 1.5).cpu().numpy()
    for world in (2, 4, 7, 16):                                  # 10 tile rows: the last ranks of 16 own nothing
        img, _ = _assemble_strips(r, cam, 1, 2, 1.5, world)
        assert np.array_equal(img, full)
    r.close()
