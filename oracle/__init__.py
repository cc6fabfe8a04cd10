"""ctypes front-end of the CPU oracle (oracle/flod_oracle.c) -- TEST INFRASTRUCTURE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package.  It imports nothing from paper_2408_12894_b200/ and the product never
imports it.
"""
from __future__ import annotations

import ctypes as C

import numpy as np

from .build import build_oracle

SKIP_THR = float(np.float32(1.0 / 255.0))   # DESIGN R11: alpha below (float)(1/255) is skipped
STOP_THR = float(np.float32(1e-4))          # DESIGN R11/R12: stop after T falls below 1e-4
ST_UNSELECTED, ST_CULL_NEAR, ST_CULL_DEAD, ST_CULL_DET, ST_EMPTY_RECT, ST_VISIBLE = range(6)


class _LevelDesc(C.Structure):
    _fields_ = [("n", C.c_int64), ("level", C.c_int), ("s_min", C.c_float),
                ("mean", C.c_void_p), ("log_scale", C.c_void_p), ("quat", C.c_void_p),
                ("opacity_logit", C.c_void_p), ("sh", C.c_void_p)]


class _Camera(C.Structure):
    _fields_ = [("R", C.c_float * 9), ("t", C.c_float * 3),
                ("fx", C.c_float), ("fy", C.c_float), ("cx", C.c_float), ("cy", C.c_float),
                ("width", C.c_int), ("height", C.c_int), ("z_near", C.c_float), ("bg", C.c_float * 3)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build_oracle())
        L.orc_scale_constraint.restype = C.c_double
        L.orc_scale_constraint.argtypes = [C.c_int, C.c_double, C.c_double, C.c_int]
        L.orc_effective_scale.restype = C.c_double
        L.orc_effective_scale.argtypes = [C.c_double, C.c_double]
        L.orc_d_proj.restype = C.c_double
        L.orc_d_proj.argtypes = [C.c_double, C.c_double, C.c_double]
        L.orc_scene_create.restype = C.c_void_p
        L.orc_scene_create.argtypes = [C.c_int, C.c_void_p, C.c_int]
        L.orc_scene_destroy.argtypes = [C.c_void_p]
        L.orc_scene_n_total.restype = C.c_int64
        L.orc_scene_n_total.argtypes = [C.c_void_p]
        for name in ("cov", "opacity", "kappa", "dead"):
            f = getattr(L, "orc_scene_" + name)
            f.restype = C.c_void_p
            f.argtypes = [C.c_void_p]
        L.orc_frame_create.restype = C.c_void_p
        L.orc_frame_create.argtypes = [C.c_void_p, C.c_void_p, C.c_int, C.c_int, C.c_float, C.c_void_p]
        L.orc_frame_create_ex.restype = C.c_void_p
        L.orc_frame_create_ex.argtypes = [C.c_void_p, C.c_void_p, C.c_int, C.c_int, C.c_float, C.c_void_p, C.c_int]
        L.orc_frame_destroy.argtypes = [C.c_void_p]
        for name in ("mask", "state", "mu2d", "depth", "cov2d", "conic", "rect", "n_tiles", "rgb",
                     "tile_start", "centre"):
            f = getattr(L, "orc_frame_" + name)
            f.restype = C.c_void_p
            f.argtypes = [C.c_void_p]
        L.orc_frame_thresholds.restype = C.c_void_p
        L.orc_frame_thresholds.argtypes = [C.c_void_p, C.c_int]
        L.orc_frame_tx.argtypes = [C.c_void_p]
        L.orc_frame_ty.argtypes = [C.c_void_p]
        L.orc_frame_counts.argtypes = [C.c_void_p, C.c_void_p]
        L.orc_frame_sorted_pairs.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.orc_frame_composite.argtypes = [C.c_void_p, C.c_double, C.c_double, C.c_int,
                                          C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.orc_frame_trace_pixel.restype = C.c_int
        L.orc_frame_trace_pixel.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_double, C.c_double,
                                            C.c_void_p, C.c_void_p, C.c_int]
        L.orc_sh_basis.argtypes = [C.c_int, C.c_void_p, C.c_void_p]
        L.orc_band_thresholds.argtypes = [C.c_int, C.c_void_p, C.c_int, C.c_int, C.c_float, C.c_float,
                                          C.c_void_p, C.c_void_p]
        L.orc_activate_one.argtypes = [C.c_void_p] * 2 + [C.c_float] + [C.c_void_p] * 4
        L.orc_num_threads.restype = C.c_int
        _lib = L
    return _lib


def _f32(a):
    return np.ascontiguousarray(a, dtype=np.float32)


def _view(ptr, shape, dtype):
    n = int(np.prod(shape))
    if n == 0:
        return np.zeros(shape, dtype=dtype)
    buf = (C.c_char * (n * np.dtype(dtype).itemsize)).from_address(ptr)
    return np.frombuffer(buf, dtype=dtype).reshape(shape).copy()   # copy: the C object may be freed first


def scale_constraint(level, tau, rho, l_max):
    return lib().orc_scale_constraint(level, tau, rho, l_max)


def effective_scale(s_opt, s_min):
    return lib().orc_effective_scale(s_opt, s_min)


def d_proj(s_min, gamma, f):
    return lib().orc_d_proj(s_min, gamma, f)


def sh_basis(degree, d):
    d = np.ascontiguousarray(d, dtype=np.float64)
    Y = np.zeros(16, dtype=np.float64)
    lib().orc_sh_basis(degree, d.ctypes.data, Y.ctypes.data)
    return Y[:(degree + 1) ** 2]


def band_thresholds(s_min, l_start, l_end, fx, gamma):
    s = _f32(s_min)
    lo = np.zeros(len(s), np.float32)
    hi = np.zeros(len(s), np.float32)
    lib().orc_band_thresholds(len(s), s.ctypes.data, l_start, l_end, float(np.float32(fx)),
                              float(np.float32(gamma)), lo.ctypes.data, hi.ctypes.data)
    return lo, hi


def activate_one(log_scale, quat, logit):
    ls, q = _f32(log_scale), _f32(quat)
    cov = np.zeros(6, np.float32)
    o = np.zeros(1, np.float32)
    k = np.zeros(1, np.float32)
    d = np.zeros(1, np.uint8)
    lib().orc_activate_one(ls.ctypes.data, q.ctypes.data, float(np.float32(logit)), cov.ctypes.data,
                           o.ctypes.data, k.ctypes.data, d.ctypes.data)
    return cov, float(o[0]), float(k[0]), bool(d[0])


def num_threads():
    return lib().orc_num_threads()


def _camera_struct(cam):
    c = _Camera()
    c.R[:] = [float(v) for v in np.asarray(cam.R, dtype=np.float32).reshape(9)]
    c.t[:] = [float(v) for v in np.asarray(cam.t, dtype=np.float32).reshape(3)]
    c.fx, c.fy, c.cx, c.cy = cam.fx, cam.fy, cam.cx, cam.cy
    c.width, c.height, c.z_near = cam.width, cam.height, cam.z_near
    c.bg[:] = [float(v) for v in cam.bg]
    return c


class OracleScene:
    """Activated multi-level scene (step O0).  `levels`: objects with the fields of flod_synth.Level."""

    def __init__(self, levels, sh_degree):
        self._keep = []
        descs = (_LevelDesc * len(levels))()
        for i, lv in enumerate(levels):
            arrs = [_f32(lv.mean), _f32(lv.log_scale), _f32(lv.quat), _f32(lv.opacity_logit), _f32(lv.sh)]
            self._keep.append(arrs)
            descs[i].n = arrs[0].shape[0]
            descs[i].level = lv.level
            descs[i].s_min = lv.s_min
            (descs[i].mean, descs[i].log_scale, descs[i].quat, descs[i].opacity_logit,
             descs[i].sh) = [a.ctypes.data for a in arrs]
        self.level_ids = [lv.level for lv in levels]
        self.s_min = [lv.s_min for lv in levels]
        self.counts = [int(np.asarray(lv.mean).shape[0]) for lv in levels]
        self.sh_degree = sh_degree
        self._h = lib().orc_scene_create(len(levels), C.addressof(descs), sh_degree)
        if not self._h:
            raise ValueError("orc_scene_create failed")
        self.n_total = lib().orc_scene_n_total(self._h)
        self._keep = None  # the C side copied what it needs

    def __del__(self):
        if getattr(self, "_h", None):
            lib().orc_scene_destroy(self._h)
            self._h = None

    @property
    def cov(self):
        return _view(lib().orc_scene_cov(self._h), (self.n_total, 6), np.float32)

    @property
    def opacity(self):
        return _view(lib().orc_scene_opacity(self._h), (self.n_total,), np.float32)

    @property
    def kappa(self):
        return _view(lib().orc_scene_kappa(self._h), (self.n_total,), np.float32)

    @property
    def dead(self):
        return _view(lib().orc_scene_dead(self._h), (self.n_total,), np.uint8)

    def frame(self, cam, l_start, l_end, gamma, ref_pos=None, geometry_only=False, fp64=False, pair_rule=1):
        return OracleFrame(self, cam, l_start, l_end, gamma, ref_pos, geometry_only, fp64, pair_rule)


class OracleFrame:
    """Steps O1-O6 for one camera and level mode; `composite` is O7.  Levels are level ids."""

    def __init__(self, scene, cam, l_start, l_end, gamma, ref_pos=None, geometry_only=False, fp64=False, pair_rule=1):
        """geometry_only: steps O1-O4 and the per-tile counts of O6 only (no colours, no stored lists, no image).
        fp64: variant O64 -- every step in fp64 with no intermediate rounding (a report, never a parity target).
        pair_rule: which tiles a visible Gaussian is listed in (DESIGN R13 / R26): 1 = every tile of its rect,
        2 = the tiles of its rect that hold a pixel centre of the padded alpha = 1/255 ellipse."""
        if pair_rule not in (1, 2) or (fp64 and pair_rule != 1):
            raise ValueError("pair_rule is 1 (box) or 2 (ellipse); O64 uses rule 1")
        self.pair_rule = pair_rule
        self.scene = scene
        self.W, self.H = cam.width, cam.height
        cs = _camera_struct(cam)
        ref = None if ref_pos is None else _f32(ref_pos)
        base = scene.level_ids[0] - 1
        self._h = lib().orc_frame_create_ex(scene._h, C.addressof(cs), l_start - base, l_end - base,
                                            float(np.float32(gamma)), None if ref is None else ref.ctypes.data,
                                            (0 if geometry_only else 3) | (4 if fp64 else 0) | (8 if pair_rule == 2 else 0))
        if not self._h:
            raise ValueError("orc_frame_create failed (bad level range or gamma)")
        self.TX, self.TY = lib().orc_frame_tx(self._h), lib().orc_frame_ty(self._h)
        cnt = np.zeros(6, np.int64)
        lib().orc_frame_counts(self._h, cnt.ctypes.data)
        self.counts = dict(zip(("n_scan", "n_sel", "n_front", "n_vis", "n_pairs", "n_bf"), map(int, cnt)))

    def __del__(self):
        if getattr(self, "_h", None):
            lib().orc_frame_destroy(self._h)
            self._h = None

    def _arr(self, name, shape, dtype):
        return _view(getattr(lib(), "orc_frame_" + name)(self._h), shape, dtype)

    n = property(lambda self: self.scene.n_total)
    mask = property(lambda self: self._arr("mask", (self.n,), np.uint8))
    state = property(lambda self: self._arr("state", (self.n,), np.uint8))
    mu2d = property(lambda self: self._arr("mu2d", (self.n, 2), np.float32))
    depth = property(lambda self: self._arr("depth", (self.n,), np.float32))
    cov2d = property(lambda self: self._arr("cov2d", (self.n, 3), np.float32))
    conic = property(lambda self: self._arr("conic", (self.n, 3), np.float32))
    rect = property(lambda self: self._arr("rect", (self.n, 4), np.int32))
    n_tiles = property(lambda self: self._arr("n_tiles", (self.n,), np.uint32))
    rgb = property(lambda self: self._arr("rgb", (self.n, 3), np.float64))
    tile_start = property(lambda self: self._arr("tile_start", (self.TX * self.TY + 1,), np.uint32))
    centre = property(lambda self: self._arr("centre", (3,), np.float32))

    @property
    def tile_counts(self):
        ts = self.tile_start.astype(np.int64)
        return (ts[1:] - ts[:-1]).astype(np.uint32)

    def thresholds(self):
        L = len(self.scene.level_ids)
        lo = _view(lib().orc_frame_thresholds(self._h, 0), (16,), np.float32)[:L].copy()
        hi = _view(lib().orc_frame_thresholds(self._h, 1), (16,), np.float32)[:L].copy()
        return lo, hi

    def sorted_pairs(self):
        P = self.counts["n_pairs"]
        tile = np.zeros(P, np.uint32)
        depth = np.zeros(P, np.float32)
        gid = np.zeros(P, np.uint32)
        lib().orc_frame_sorted_pairs(self._h, tile.ctypes.data, depth.ctypes.data, gid.ctypes.data)
        return tile, depth, gid

    def composite(self, skip_thr=SKIP_THR, stop_thr=STOP_THR, brute=False, stats=False):
        out = np.zeros((3, self.H, self.W), np.float64)
        if stats:
            E = np.zeros((self.H, self.W), np.uint32)
            B = np.zeros((self.H, self.W), np.uint32)
            T = np.zeros((self.H, self.W), np.float64)
            lib().orc_frame_composite(self._h, skip_thr, stop_thr, int(brute), out.ctypes.data,
                                      E.ctypes.data, B.ctypes.data, T.ctypes.data)
            return out, E, B, T
        lib().orc_frame_composite(self._h, skip_thr, stop_thr, int(brute), out.ctypes.data, None, None, None)
        return out

    def trace_pixel(self, i, j, skip_thr=SKIP_THR, stop_thr=STOP_THR, cap=4096):
        a = np.zeros(cap, np.float64)
        t = np.zeros(cap, np.float64)
        n = lib().orc_frame_trace_pixel(self._h, i, j, skip_thr, stop_thr, a.ctypes.data, t.ctypes.data, cap)
        n = min(n, cap)
        return a[:n], t[:n]
