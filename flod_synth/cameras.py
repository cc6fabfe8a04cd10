"""Pinhole cameras and the pose trajectories of the benchmark configs.

Camera convention (include/flod.h: flod_camera): x_cam = R x_world + t, camera axes +x right,
+y down, +z forward; fx = fy = (W/2)/tan(30 deg) (horizontal FoV 60 deg), principal point at the
image centre, z_near = 0.2, black background.  Look-at: right = normalise(fwd x up),
down = fwd x right, R rows = (right, down, fwd), t = -R eye, world up = (0,1,0).
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np


@dataclass
class Camera:
    R: np.ndarray            # [3,3] fp32 row-major
    t: np.ndarray            # [3] fp32
    fx: float
    fy: float
    cx: float
    cy: float
    width: int
    height: int
    z_near: float = 0.2
    bg: tuple = (0.0, 0.0, 0.0)
    eye: np.ndarray = field(default=None, repr=False)   # fp64 eye the pose was built from (info only)


def look_at(eye, target, up=(0.0, 1.0, 0.0)):
    eye = np.asarray(eye, dtype=np.float64)
    fwd = np.asarray(target, dtype=np.float64) - eye
    fwd /= np.linalg.norm(fwd)
    right = np.cross(fwd, np.asarray(up, dtype=np.float64))
    right /= np.linalg.norm(right)
    down = np.cross(fwd, right)
    R = np.stack([right, down, fwd])
    t = -R @ eye
    return R, t


def pinhole(R, t, width, height, eye=None, fov_deg=60.0, z_near=0.2, bg=(0.0, 0.0, 0.0)) -> Camera:
    f = (width / 2.0) / math.tan(math.radians(fov_deg / 2.0))
    f32 = lambda v: float(np.float32(v))
    return Camera(R=np.ascontiguousarray(R, dtype=np.float32), t=np.ascontiguousarray(t, dtype=np.float32),
                  fx=f32(f), fy=f32(f), cx=f32(width / 2.0), cy=f32(height / 2.0),
                  width=int(width), height=int(height), z_near=f32(z_near), bg=tuple(f32(b) for b in bg),
                  eye=None if eye is None else np.asarray(eye, dtype=np.float64))


def make_poses(config: int, width: int | None = None, height: int | None = None, n_poses: int | None = None):
    """The pose list of BASELINE.json `configs[config]` (config 2 shares config 1's)."""
    if config == 2:
        config = 1
    cams = []
    if config == 0:
        W, H = (width or 128), (height or 128)
        eye = (0.0, 0.0, -3.0)
        R, t = look_at(eye, (0.0, 0.0, 0.0))
        return [pinhole(R, t, W, H, eye=eye)]
    if config == 1:
        W, H, n = (width or 1237), (height or 822), (n_poses or 200)
        for k in range(n):
            th = 2.0 * math.pi * k / n
            eye = (12.0 * math.cos(th), 2.0, 8.0 * math.sin(th))
            R, t = look_at(eye, (0.0, 0.0, 0.0))
            cams.append(pinhole(R, t, W, H, eye=eye))
        return cams
    if config == 3:
        W, H, n = (width or 980), (height or 545), (n_poses or 150)
        for k in range(n):
            th = 2.0 * math.pi * k / n
            eye = (6.0 * math.cos(th), 1.5, 6.0 * math.sin(th))
            R, t = look_at(eye, (0.0, 0.0, 0.0))
            cams.append(pinhole(R, t, W, H, eye=eye))
        return cams
    if config == 4:
        W, H, n = (width or 960), (height or 540), (n_poses or 300)
        for k in range(n):
            eye = np.array([-45.0 + 50.0 * k / max(n - 1, 1), 3.0, 0.0])
            yaw = math.radians(10.0) * math.sin(2.0 * math.pi * k / 100.0)
            fwd = np.array([math.cos(yaw), 0.0, math.sin(yaw)])
            R, t = look_at(eye, eye + fwd)
            cams.append(pinhole(R, t, W, H, eye=eye))
        return cams
    raise ValueError(f"no pose recipe for config {config}")


def poses_checksum(cams) -> str:
    """sha256 over the fp32 fields of a pose list (R, t, fx, fy, cx, cy, width, height, z_near)."""
    import hashlib
    h = hashlib.sha256()
    for c in cams:
        h.update(np.ascontiguousarray(c.R, dtype=np.float32).tobytes()); h.update(np.ascontiguousarray(c.t, dtype=np.float32).tobytes())
        h.update(np.array([c.fx, c.fy, c.cx, c.cy, c.z_near], dtype=np.float32).tobytes())
        h.update(np.array([c.width, c.height], dtype=np.int32).tobytes())
    return h.hexdigest()
