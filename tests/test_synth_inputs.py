"""The seeded input generators (flod_synth) produce the scenes and poses whose checksums are committed under
tests/golden/scene_checksums.json (written by tests/golden/make_scene_checksums.py): a numpy or platform change that
silently alters a "seeded" scene shows up here, not as an unexplained change of every measured number."""
import json
import os

import numpy as np
import pytest

import flod_synth as fs

GOLD = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "scene_checksums.json")))


@pytest.mark.parametrize("config", [0, 1, 3, 4])
def test_scaled_scene_checksums(config):
    assert fs.scene_checksum(fs.make_scene(config, count_scale=0.01)) == GOLD["scaled"][str(config)]


def test_config0_full_scene_and_pose_checksums():
    assert fs.scene_checksum(fs.make_scene(0)) == GOLD["full"]["0"]
    for config in (0, 1, 3, 4):
        assert fs.poses_checksum(fs.make_poses(config)) == GOLD["poses"][str(config)]
    assert fs.poses_checksum(fs.make_poses(4, 1920, 1080)) == GOLD["poses"]["4@1920x1080"]


def test_scene_shapes_follow_baseline_configs():
    """BASELINE.json configs: per-level counts, SH degree, image sizes, pose counts; Eq. 3 ladder (floor halves per
    level from 0.2, top level 0); stored scale = exp(s_opt) + s_min >= s_min (Eq. 4)."""
    for config, counts in ((1, [50_000, 200_000, 600_000, 1_500_000, 3_000_000]), (3, [30_000, 120_000, 400_000, 900_000, 1_800_000]),
                           (4, [200_000, 800_000, 2_000_000, 4_000_000, 8_000_000])):
        assert fs.scene_spec(config)["counts"] == counts and fs.scene_spec(config)["sh_degree"] == 3
        sc = fs.make_scene(config, count_scale=0.001)
        assert [lv.s_min for lv in sc.levels] == [float(np.float32(0.2 * 2.0 ** (1 - l))) for l in range(1, 5)] + [0.0]
        for lv in sc.levels:
            assert lv.sh.shape[1:] == (16, 3) and (np.exp(lv.log_scale.astype(np.float64)) >= lv.s_min * (1 - 1e-6)).all()
    assert [(c.width, c.height) for c in (fs.make_poses(1)[0], fs.make_poses(3)[0], fs.make_poses(4)[0])] == [(1237, 822), (980, 545), (960, 540)]
    assert (len(fs.make_poses(1)), len(fs.make_poses(3)), len(fs.make_poses(4))) == (200, 150, 300)
