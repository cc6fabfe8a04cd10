"""Seeded multi-level Gaussian scenes shaped like the paper's workloads.

The per-level counts imitate the paper's 10K/33K/409K/979K/2017K ladder and the
image sizes its datasets.  Every array is fp32, C-contiguous, and laid out as
`include/flod.h: flod_level_desc` expects.  A level stores the log of the EFFECTIVE scale
s^(l) = exp(s_opt) + s_min^(l) (Eq. 4; saved clones hold S^(l));
`s_min` travels beside it as metadata for Eq. 7.

Draw order per level (fixed, so a seed names one scene): positions, s_opt, quaternions, opacity
logits, SH.  Generator: numpy PCG64 `default_rng(1000*config + level)`; cluster layout uses
`default_rng(1000*config + 900)`.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

SH_Y0 = 0.5 * math.sqrt(1.0 / math.pi)  # only used to store "RGB" as a DC coefficient (config 0)


@dataclass
class Level:
    level: int              # 1-based
    s_min: float            # Eq. 3 value for this level (0 at the top level)
    mean: np.ndarray        # [n,3]
    log_scale: np.ndarray   # [n,3] log of effective scale
    quat: np.ndarray        # [n,4] w,x,y,z (unit here, any non-zero norm is legal)
    opacity_logit: np.ndarray  # [n]
    sh: np.ndarray          # [n,K,3]

    @property
    def n(self) -> int:
        return int(self.mean.shape[0])


@dataclass
class Scene:
    config: int
    sh_degree: int
    levels: list = field(default_factory=list)

    @property
    def n_total(self) -> int:
        return sum(l.n for l in self.levels)

    @property
    def offsets(self):
        off = [0]
        for l in self.levels:
            off.append(off[-1] + l.n)
        return off


SCENE_SPECS = {
    # config: counts per level, sh degree, image sizes, number of poses
    0: dict(counts=[1_000, 4_000], sh_degree=0, images=[(128, 128)], n_poses=1),
    1: dict(counts=[50_000, 200_000, 600_000, 1_500_000, 3_000_000], sh_degree=3,
            images=[(1237, 822)], n_poses=200),
    3: dict(counts=[30_000, 120_000, 400_000, 900_000, 1_800_000], sh_degree=3,
            images=[(980, 545)], n_poses=150),
    4: dict(counts=[200_000, 800_000, 2_000_000, 4_000_000, 8_000_000], sh_degree=3,
            images=[(960, 540), (1920, 1080)], n_poses=300),
}
SCENE_SPECS[2] = SCENE_SPECS[1]  # config 2 = config 1's scene and poses, other render modes


def scene_spec(config: int) -> dict:
    return SCENE_SPECS[config]


def _unit_rows(a: np.ndarray) -> np.ndarray:
    return a / np.linalg.norm(a, axis=1, keepdims=True)


def _positions_outdoor(rng, n, layout):
    n_c = int(0.7 * n)
    n_s = n - n_c
    idx = rng.integers(0, layout["centres"].shape[0], n_c)
    pc = layout["centres"][idx] + rng.normal(0.0, 2.0, (n_c, 3))
    d = _unit_rows(rng.normal(size=(n_s, 3)))
    ps = d * rng.uniform(16.0, 20.0, (n_s, 1))
    return np.concatenate([pc, ps])


def _positions_object(rng, n, layout):
    n_o = int(0.8 * n)
    n_b = n - n_o
    d = _unit_rows(rng.normal(size=(n_o, 3)))
    po = d * (3.0 + rng.normal(0.0, 0.1, (n_o, 1)))
    db = _unit_rows(rng.normal(size=(n_b, 3)))
    pb = db * (30.0 * rng.uniform(0.0, 1.0, (n_b, 1)) ** (1.0 / 3.0))  # uniform in the ball
    return np.concatenate([po, pb])


def _positions_large(rng, n, layout):
    k = layout["centres"].shape[0]
    idx = rng.integers(0, k, n)
    e = rng.normal(size=(n, 3)) * layout["sigma"][idx]
    c, s = np.cos(layout["yaw"][idx]), np.sin(layout["yaw"][idx])
    x = c * e[:, 0] + s * e[:, 2]
    z = -s * e[:, 0] + c * e[:, 2]
    return layout["centres"][idx] + np.stack([x, e[:, 1], z], axis=1)


def _layout(config: int):
    rng = np.random.default_rng(1000 * config + 900)
    if config in (1, 2):
        return dict(centres=rng.uniform(-1.0, 1.0, (64, 3)) * np.array([10.0, 3.0, 10.0]))
    if config == 4:
        lo = np.array([-50.0, 0.0, -50.0])
        hi = np.array([50.0, 20.0, 50.0])
        centres = rng.uniform(lo, hi, (200, 3))
        sigma = np.stack([rng.uniform(1.0, 8.0, 200), rng.uniform(0.5, 3.0, 200),
                          rng.uniform(1.0, 8.0, 200)], axis=1)
        yaw = rng.uniform(0.0, 2.0 * math.pi, 200)
        return dict(centres=centres, sigma=sigma, yaw=yaw)
    return {}


def make_scene(config: int, count_scale: float = 1.0, levels: list | None = None) -> Scene:
    """Build the scene of BASELINE.json `configs[config]`.

    count_scale < 1 shrinks every level's count (CPU-sized parity cases keep the distribution).
    `levels` (1-based) restricts which levels are generated; the others stay in the ladder but are
    returned empty-free, i.e. simply absent - callers that upload must pass consecutive levels.
    """
    if config == 2:
        config = 1
    spec = SCENE_SPECS[config]
    counts = [max(1, int(round(c * count_scale))) for c in spec["counts"]]
    L = len(counts)
    layout = _layout(config)
    scene = Scene(config=config, sh_degree=spec["sh_degree"])
    K = (spec["sh_degree"] + 1) ** 2
    for l in range(1, L + 1):
        if levels is not None and l not in levels:
            continue
        n = counts[l - 1]
        rng = np.random.default_rng(1000 * config + l)
        if config == 0:
            mean = rng.uniform(-1.0, 1.0, (n, 3))
            lo, hi = ((-2.5, -1.5), (-4.0, -2.5))[l - 1]
            log_scale = rng.uniform(lo, hi, (n, 3))
            s_min = (0.027, 0.0)[l - 1]
            quat = _unit_rows(rng.normal(size=(n, 4)))
            logit = rng.normal(0.0, 1.0, n)
            rgb = rng.uniform(0.0, 1.0, (n, 1, 3))
            sh = (rgb - 0.5) / SH_Y0
        else:
            pos_fn = {1: _positions_outdoor, 3: _positions_object, 4: _positions_large}[config]
            mean = pos_fn(rng, n, layout)
            floor = 0.2 * 2.0 ** (1 - l)
            s_min = floor if l < L else 0.0
            s_opt = math.log(floor) + rng.normal(0.0, 1.0, (n, 3))
            log_scale = np.log(np.exp(s_opt) + s_min)          # Eq. 4, stored as effective scale
            quat = _unit_rows(rng.normal(size=(n, 4)))
            logit = rng.normal(0.0, 1.5, n)
            sh = rng.standard_normal((n, K, 3), dtype=np.float32)
            sh[:, 0, :] = 0.5 + 0.2 * sh[:, 0, :]
            sh[:, 1:, :] *= 0.05
        scene.levels.append(Level(
            level=l, s_min=float(np.float32(s_min)),
            mean=np.ascontiguousarray(mean, dtype=np.float32),
            log_scale=np.ascontiguousarray(log_scale, dtype=np.float32),
            quat=np.ascontiguousarray(quat, dtype=np.float32),
            opacity_logit=np.ascontiguousarray(logit, dtype=np.float32),
            sh=np.ascontiguousarray(sh, dtype=np.float32)))
    return scene


def make_random_scene(seed: int, n_per_level=(200, 300), s_min=(0.05, 0.0), sh_degree: int = 0,
                      extent: float = 1.0, log_scale_range=(-3.5, -1.5)) -> Scene:
    """Small free-form scene for property tests (brute-force oracle equivalence and the like)."""
    rng = np.random.default_rng(seed)
    K = (sh_degree + 1) ** 2
    scene = Scene(config=-1, sh_degree=sh_degree)
    for i, n in enumerate(n_per_level):
        sh = rng.normal(0.0, 0.3, (n, K, 3))
        sh[:, 0, :] += 0.5
        scene.levels.append(Level(
            level=i + 1, s_min=float(np.float32(s_min[i])),
            mean=rng.uniform(-extent, extent, (n, 3)).astype(np.float32),
            log_scale=rng.uniform(*log_scale_range, (n, 3)).astype(np.float32),
            quat=_unit_rows(rng.normal(size=(n, 4))).astype(np.float32),
            opacity_logit=rng.normal(0.0, 1.5, n).astype(np.float32),
            sh=np.ascontiguousarray(sh, dtype=np.float32)))
    return scene


def scene_checksum(scene: Scene) -> str:
    """sha256 over every level's id, s_min and arrays (bytes, in field order): names the exact inputs a seed produced,
    so that a numpy / platform change that alters a "seeded" scene is noticed (tests/golden/scene_checksums.json)."""
    import hashlib
    h = hashlib.sha256()
    h.update(np.int32(scene.sh_degree).tobytes())
    for lv in scene.levels:
        h.update(np.int32(lv.level).tobytes()); h.update(np.float32(lv.s_min).tobytes())
        for a in (lv.mean, lv.log_scale, lv.quat, lv.opacity_logit, lv.sh):
            h.update(np.ascontiguousarray(a, dtype=np.float32).tobytes())
    return h.hexdigest()
