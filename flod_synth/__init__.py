"""Seeded synthetic inputs (scenes, cameras) shared by the oracle tests, the GPU tests and bench.py.

This package holds input generation only: none of the renderer's arithmetic lives here, and neither
`oracle/` nor `paper_2408_12894_b200/` is imported from it.  The recipes are those of DESIGN.md §4
(SURVEY.md §8(d)); they stand in for the paper's datasets, which are not available.
"""
from .scenes import Level, Scene, make_scene, scene_checksum, scene_spec, SCENE_SPECS
from .cameras import Camera, look_at, make_poses, pinhole, poses_checksum

__all__ = ["Level", "Scene", "make_scene", "scene_checksum", "scene_spec", "SCENE_SPECS",
           "Camera", "look_at", "make_poses", "pinhole", "poses_checksum"]
