"""Small builders shared by the tests: hand-made levels and cameras (inputs only, no method arithmetic)."""
from __future__ import annotations

import math
from types import SimpleNamespace

import numpy as np

Y0 = 0.5 * math.sqrt(1.0 / math.pi)


def level(level_id, s_min, mean, scale, quat=None, opacity=None, rgb=None, sh=None, logit=None):
    """One level from plain values: `scale` is the effective scale (world units), `opacity` in (0,1)."""
    mean = np.atleast_2d(np.asarray(mean, dtype=np.float64))
    n = mean.shape[0]
    scale = np.broadcast_to(np.asarray(scale, dtype=np.float64), (n, 3)) if np.ndim(scale) < 2 else np.asarray(scale)
    quat = np.tile([1.0, 0.0, 0.0, 0.0], (n, 1)) if quat is None else np.atleast_2d(np.asarray(quat, dtype=np.float64))
    if logit is None:
        opacity = np.full(n, 0.5) if opacity is None else np.broadcast_to(np.asarray(opacity, dtype=np.float64), (n,))
        logit = np.log(opacity / (1.0 - opacity))
    else:
        logit = np.broadcast_to(np.asarray(logit, dtype=np.float64), (n,))
    if sh is None:
        rgb = np.full((n, 3), 0.5) if rgb is None else np.broadcast_to(np.asarray(rgb, dtype=np.float64), (n, 3))
        sh = ((rgb - 0.5) / Y0).reshape(n, 1, 3)
    return SimpleNamespace(level=level_id, s_min=float(np.float32(s_min)),
                           mean=mean.astype(np.float32), log_scale=np.log(scale).astype(np.float32),
                           quat=quat.astype(np.float32), opacity_logit=np.asarray(logit).astype(np.float32),
                           sh=np.ascontiguousarray(sh, dtype=np.float32))


def camera(width=33, height=33, f=100.0, R=None, t=None, z_near=0.2, bg=(0.0, 0.0, 0.0), cx=None, cy=None, fy=None):
    """Identity pose by default: camera at the origin looking down +z, +x right, +y down.  f is fx; fy defaults to it."""
    return SimpleNamespace(R=np.eye(3, dtype=np.float32) if R is None else np.asarray(R, dtype=np.float32),
                           t=np.zeros(3, dtype=np.float32) if t is None else np.asarray(t, dtype=np.float32),
                           fx=float(np.float32(f)), fy=float(np.float32(f if fy is None else fy)),
                           cx=float(np.float32(width / 2.0 if cx is None else cx)),
                           cy=float(np.float32(height / 2.0 if cy is None else cy)),
                           width=width, height=height, z_near=float(np.float32(z_near)), bg=tuple(bg))


def random_rotation(rng):
    q = rng.normal(size=4)
    q /= np.linalg.norm(q)
    w, x, y, z = q
    return np.array([[1 - 2 * (y * y + z * z), 2 * (x * y - w * z), 2 * (x * z + w * y)],
                     [2 * (x * y + w * z), 1 - 2 * (x * x + z * z), 2 * (y * z - w * x)],
                     [2 * (x * z - w * y), 2 * (y * z + w * x), 1 - 2 * (x * x + y * y)]]), q
