"""Writes tests/golden/scene_checksums.json: sha256 of every synthetic scene and pose list the tests and bench.py use
(flod_synth only -- no oracle, no CUDA path).  Run once per change of the recipe in DESIGN.md §4:

    python tests/golden/make_scene_checksums.py

"full" entries are BASELINE.json's sizes (checked on the GPU box, where the scenes are built anyway); "scaled" entries
are the same recipes at count_scale = 0.01 (checked by the CPU suite in a second)."""
import json
import os
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))

import numpy as np

import flod_synth as fs

out = {"numpy": np.__version__, "full": {}, "scaled": {}, "poses": {}}
for config in (0, 1, 3, 4):
    out["full"][str(config)] = fs.scene_checksum(fs.make_scene(config))
    out["scaled"][str(config)] = fs.scene_checksum(fs.make_scene(config, count_scale=0.01))
    out["poses"][str(config)] = fs.poses_checksum(fs.make_poses(config))
out["poses"]["4@1920x1080"] = fs.poses_checksum(fs.make_poses(4, 1920, 1080))
json.dump(out, open(os.path.join(HERE, "scene_checksums.json"), "w"), indent=1)
print(json.dumps(out, indent=1))
