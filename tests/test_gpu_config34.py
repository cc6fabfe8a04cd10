"""Parity at full size on BASELINE.json configs[3] (object-centric scene, 3.25M Gaussians, 980x545, every level alone) and
configs[4] (large scene, 15M Gaussians, selective {2,3,4} and {3,4,5} at gamma = 1 px, 960x540 and 1920x1080), in the
launch configuration bench.py times.  Per mode, three poses: selection masks, frame counters, per-tile pair counts, the
projected records and the whole sorted (tile, depth, gid) sequence exactly; the full image (1e-3 with the envelope rule
of DESIGN §3) on one pose per mode.  Scenes are uploaded once per module."""
import gc

import numpy as np
import pytest

import flod_synth as fs
from oracle import OracleScene
from test_gpu_parity import check_frame

pytestmark = pytest.mark.gpu

MAX_PAIRS = 32 << 20      # bench.py's workspace


def _report_checksum(config, scene):
    """Full-size scene against tests/golden/scene_checksums.json.  Reported, not asserted: parity does not depend on it
    (oracle and CUDA path read the same arrays), and numpy's SIMD paths for exp / log may differ between host CPUs."""
    import json, os
    gold = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "scene_checksums.json")))["full"][str(config)]
    got = fs.scene_checksum(scene)
    print(f"config {config} scene checksum {'matches' if got == gold else 'DIFFERS from'} tests/golden/scene_checksums.json ({got[:16]})")


def _setup(config, width, height):
    from paper_2408_12894_b200 import build
    build.build()
    import paper_2408_12894_b200 as pkg
    scene = fs.make_scene(config)
    _report_checksum(config, scene)
    osc = OracleScene(scene.levels, scene.sh_degree)
    r = pkg.Renderer(0)
    r.upload_levels(scene.levels, scene.sh_degree)
    r.set_workspace(width, height, MAX_PAIRS)
    r.set_options(pkg.FLOD_OPT_DEBUG)
    r.set_pair_rule(pkg.PAIR_RULE_ELLIPSE if config == 3 else pkg.PAIR_RULE_BOX)     # the rule that pays on each config
    return scene, osc, r


@pytest.fixture(scope="module")
def config3():
    scene, osc, r = _setup(3, 980, 545)
    yield scene, fs.make_poses(3), osc, r
    r.close()
    del osc, scene
    gc.collect()


@pytest.mark.parametrize("l", [1, 2, 3, 4, 5])
def test_config3_single_level(config3, l):
    """Each level alone (BASELINE.json configs[3]): l = 1..3 are the frames of 13-19M pairs whose tile lists hold
    6-9K keys at clustered depths (the object's shell): k_duplicate_shared and the sliced tile sort."""
    scene, cams, osc, r = config3
    for pose in (0, 61, 122):
        res, _, fr = check_frame(r, osc, cams[pose], l, l, 1.0, image=(pose == 61))
        if res is not None:
            print(f"config3 level {l} pose {pose}: P={fr.counts['n_pairs']} n_vis={fr.counts['n_vis']} "
                  f"max list={int(fr.tile_counts.max())} max|gpu-oracle|={res[0]:.2e} marginal={res[1]}")
    assert fr.counts["n_scan"] == scene.levels[l - 1].n
    # the frame as bench.py renders it (no debug view: blend-driven ordering of the long lists) is the same image, bit for bit
    import paper_2408_12894_b200 as pkg
    dbg = r.render(cams[61], l, l, 1.0).cpu().numpy()
    r.set_options(0)
    try:
        assert np.array_equal(r.render(cams[61], l, l, 1.0).cpu().numpy(), dbg)
    finally:
        r.set_options(pkg.FLOD_OPT_DEBUG)
    if l == 3:      # the box rule (R13) on the heaviest frame of the config
        r.set_pair_rule(pkg.PAIR_RULE_BOX)
        try:
            _, _, fr1 = check_frame(r, osc, cams[61], l, l, 1.0, image=False)
        finally:
            r.set_pair_rule(pkg.PAIR_RULE_ELLIPSE)
        print(f"config3 level 3 pose 61: P box rule {fr1.counts['n_pairs']}, ellipse rule {fr.counts['n_pairs']}")


@pytest.fixture(scope="module")
def config4():
    scene, osc, r = _setup(4, 1920, 1080)
    yield scene, osc, r
    r.close()
    del osc, scene
    gc.collect()


@pytest.mark.parametrize("size", [(960, 540), (1920, 1080)])
@pytest.mark.parametrize("levels", [(2, 4), (3, 5)])
def test_config4_selective(config4, size, levels):
    """Selective rendering with levels {2,3,4} and {3,4,5} at gamma = 1 px on the 15M-Gaussian scene, both image sizes
    (8160 tiles at 1920x1080): several levels of the range contribute, and everything checked is exact."""
    scene, osc, r = config4
    cams = fs.make_poses(4, *size)
    off = scene.offsets
    for pose in (0, 149, 299):
        res, _, fr = check_frame(r, osc, cams[pose], levels[0], levels[1], 1.0, image=(pose == 149))
        per_level = [int(fr.mask[off[l]:off[l + 1]].sum()) for l in range(5)]
        assert sum(n > 0 for n in per_level) >= 2 and all(per_level[l] == 0 for l in range(5) if not levels[0] <= l + 1 <= levels[1])
        assert sum(per_level) == fr.counts["n_sel"] and fr.TX * fr.TY == ((size[0] + 15) // 16) * ((size[1] + 15) // 16)
        if res is not None:
            print(f"config4 {size[0]}x{size[1]} levels {levels} pose {pose}: n_sel={fr.counts['n_sel']} per level {per_level} "
                  f"P={fr.counts['n_pairs']} max|gpu-oracle|={res[0]:.2e} marginal={res[1]}")


def test_config4_materialised_subset_on_the_walk(config4):
    """The paper's runtime for long trajectories on the config that needs it: G_sel {3,4,5} materialised at
    pose 100, reused at pose 110 (stale reference = the oracle's ref_pos reading, R2)."""
    scene, osc, r = config4
    cams = fs.make_poses(4, 960, 540)
    R = np.asarray(cams[100].R, np.float64).reshape(3, 3); t = np.asarray(cams[100].t, np.float64)
    c100 = np.array([-((R[0, i] * t[0] + R[1, i] * t[1]) + R[2, i] * t[2]) for i in range(3)]).astype(np.float32)
    r.subset_set_arena(3, 5)
    r.subset_build(c100, cams[100].fx, 1.0)
    n_sel = r.subset_swap()
    for pose, ref in ((100, None), (110, c100)):
        img = r.render_subset(cams[pose]).cpu().numpy()
        st = r.get_stats()
        fr = osc.frame(cams[pose], 3, 5, 1.0, ref_pos=ref, geometry_only=True, pair_rule=r.pair_rule)
        c = fr.counts
        assert n_sel == c["n_sel"] == st["n_sel"] and (st["n_front"], st["n_vis"], st["n_pairs"]) == (c["n_front"], c["n_vis"], c["n_pairs"])
        assert np.array_equal(r.debug_mask(), fr.mask)
        assert np.array_equal(r.debug_tile_counts(fr.TX * fr.TY), fr.tile_counts)
        r.set_selection_reference(ref)
        try:
            fused = r.render(cams[pose], 3, 5, 1.0).cpu().numpy()
        finally:
            r.set_selection_reference(None)
        assert np.array_equal(img, fused)


def test_config4_1080p_row_sharded_over_four_ranks(config4):
    """Screen-space sharding on the config it is meant for: 1920x1080, selective {3,4,5}: the strips four
    ranks would render, stacked the way the all-gather stacks them, are the single-GPU image bit for bit."""
    from test_gpu_parity import _assemble_strips
    scene, osc, r = config4
    cam = fs.make_poses(4, 1920, 1080)[149]
    full = r.render(cam, 3, 5, 1.0).cpu().numpy()
    st = r.get_stats()
    img, pairs = _assemble_strips(r, cam, 3, 5, 1.0, 4)
    assert np.array_equal(img, full) and pairs == st["n_pairs"]
