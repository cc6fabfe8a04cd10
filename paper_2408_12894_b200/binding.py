"""ctypes binding of libflod.so -- argument marshalling only (include/flod.h is the contract).

PyTorch appears here for device memory and streams and nothing else: the scene arena, the workspace and the
output image are torch tensors whose `data_ptr()` is handed to the C ABI; every step of the path runs in the
library's kernels.  If the library is missing this module raises -- there is no fallback.
"""
from __future__ import annotations

import ctypes as C
import os
import re

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libflod.so")
HEADER = os.path.join(HERE, "..", "include", "flod.h")

FLOD_OPT_DEBUG, FLOD_OPT_PROFILE, FLOD_OPT_COUNT, FLOD_OPT_SMALL_WINDOWS, FLOD_OPT_FULL_SORT = 1, 2, 4, 8, 16
FLOD_DBG_MASK, FLOD_DBG_TILE_COUNTS, FLOD_DBG_PROJECTED, FLOD_DBG_SORTED_PAIRS, FLOD_DBG_ACTIVATED = range(5)
PAIR_RULE_BOX, PAIR_RULE_ELLIPSE = 1, 2
FLOD_N_STAGES = 5
STAGE_NAMES = ("geometry", "colour", "duplicate", "tile_sort", "blend")
ERRORS = {-1: "FLOD_E_INVALID_ARG", -2: "FLOD_E_LEVEL_RANGE", -3: "FLOD_E_NOT_UPLOADED",
          -4: "FLOD_E_ARENA_TOO_SMALL", -5: "FLOD_E_CAPACITY", -6: "FLOD_E_CUDA", -7: "FLOD_E_NO_WORKSPACE",
          -8: "FLOD_E_STATIC_LIMIT"}


class FlodError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"{ERRORS.get(code, code)}: {msg}")
        self.code = code


class LevelDesc(C.Structure):
    _fields_ = [("n", C.c_int64), ("level", C.c_int), ("s_min", C.c_float),
                ("mean", C.c_void_p), ("log_scale", C.c_void_p), ("quat", C.c_void_p),
                ("opacity_logit", C.c_void_p), ("sh", C.c_void_p)]


class CameraStruct(C.Structure):
    _fields_ = [("R", C.c_float * 9), ("t", C.c_float * 3),
                ("fx", C.c_float), ("fy", C.c_float), ("cx", C.c_float), ("cy", C.c_float),
                ("width", C.c_int), ("height", C.c_int), ("z_near", C.c_float), ("bg", C.c_float * 3)]


class Grads(C.Structure):
    _fields_ = [("d_mean", C.c_void_p), ("d_log_scale", C.c_void_p), ("d_quat", C.c_void_p),
                ("d_opacity_logit", C.c_void_p), ("d_sh", C.c_void_p)]


class LevelMode(C.Structure):
    _fields_ = [("l_start", C.c_int), ("l_end", C.c_int)]


class Stats(C.Structure):
    _fields_ = [("n_scan", C.c_int64), ("n_sel", C.c_int64), ("n_front", C.c_int64), ("n_vis", C.c_int64),
                ("n_pairs", C.c_int64), ("max_pairs", C.c_int64), ("overflow", C.c_int),
                ("evals", C.c_int64), ("blends", C.c_int64),
                ("ms_stage", C.c_float * FLOD_N_STAGES), ("ms_total", C.c_float)]


DBG_PROJECTED_DTYPE = np.dtype([("gid", np.uint32), ("mu2d", np.float32, 2), ("depth", np.float32),
                                ("conic", np.float32, 3), ("opacity", np.float32), ("rgb", np.float32, 3),
                                ("rect", np.int32, 4)])
DBG_PAIR_DTYPE = np.dtype([("tile", np.uint32), ("depth", np.float32), ("gid", np.uint32)])


def abi_symbols():
    """Names of the functions include/flod.h declares."""
    text = open(HEADER).read()
    return re.findall(r"FLOD_API\s+[\w\s\*]+?\b(flod_\w+)\s*\(", text)


_lib = None


def load_library():
    """dlopen libflod.so and declare the prototypes.  Raises if it has not been built."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise RuntimeError(f"{LIB_PATH} is missing: build it with `python -m paper_2408_12894_b200.build` "
                           "(there is no CPU fallback)")
    L = C.CDLL(LIB_PATH)
    vp, i64, sz = C.c_void_p, C.c_int64, C.c_size_t
    L.flod_create.argtypes = [C.POINTER(vp), C.c_int]
    L.flod_destroy.argtypes = [vp]
    L.flod_scene_bytes.restype = sz
    L.flod_scene_bytes.argtypes = [C.c_int, C.POINTER(LevelDesc), C.c_int]
    L.flod_upload_levels.argtypes = [vp, C.c_int, C.POINTER(LevelDesc), C.c_int, vp, sz, vp]
    L.flod_workspace_bytes.restype = sz
    L.flod_workspace_bytes.argtypes = [vp, C.c_int, C.c_int, i64]
    L.flod_set_workspace.argtypes = [vp, vp, sz, C.c_int, C.c_int, i64]
    L.flod_set_selection_reference.argtypes = [vp, C.POINTER(C.c_float)]
    L.flod_set_options.argtypes = [vp, C.c_uint]
    L.flod_set_pair_rule.argtypes = [vp, C.c_int]
    L.flod_render.argtypes = [vp, C.POINTER(CameraStruct), LevelMode, C.c_float, vp, vp]
    L.flod_render_rows.argtypes = [vp, C.POINTER(CameraStruct), LevelMode, C.c_float, C.c_int, C.c_int, vp, vp]
    L.flod_render_to_host.argtypes = [vp, C.POINTER(CameraStruct), LevelMode, C.c_float, vp, vp]
    L.flod_render_to_host_async.argtypes = [vp, C.POINTER(CameraStruct), LevelMode, C.c_float, vp, vp, vp]
    L.flod_wait_host.argtypes = [vp]
    L.flod_subset_bytes.restype = sz
    L.flod_subset_bytes.argtypes = [vp, LevelMode]
    L.flod_subset_set_arena.argtypes = [vp, vp, sz, LevelMode]
    L.flod_subset_build.argtypes = [vp, C.POINTER(C.c_float), C.c_float, C.c_float, vp]
    L.flod_subset_ready.argtypes = [vp]
    L.flod_subset_swap.argtypes = [vp, C.POINTER(i64)]
    L.flod_render_subset.argtypes = [vp, C.POINTER(CameraStruct), vp, vp]
    L.flod_get_stats.argtypes = [vp, C.POINTER(Stats)]
    L.flod_debug_copy.argtypes = [vp, C.c_int, vp, sz]
    L.flod_launches_per_frame.argtypes = [vp]
    L.flod_backward_workspace_bytes.restype = sz
    L.flod_backward_workspace_bytes.argtypes = [vp]
    L.flod_render_backward.argtypes = [vp, C.POINTER(CameraStruct), vp, C.POINTER(Grads), vp, sz, vp]
    L.flod_overlap_prune_workspace_bytes.restype = sz
    L.flod_overlap_prune_workspace_bytes.argtypes = [i64]
    L.flod_overlap_prune.argtypes = [vp, i64, C.c_float, C.POINTER(C.c_float), vp, vp, vp, sz, vp]
    L.flod_overlap_prune_static_max_n.restype = i64
    L.flod_overlap_prune_static_max_n.argtypes = []
    L.flod_overlap_prune_static_setup.argtypes = []
    L.flod_overlap_prune_static.argtypes = [vp, i64, C.c_float, C.POINTER(C.c_float), vp, vp, vp]
    L.flod_last_error.restype = C.c_char_p
    L.flod_last_error.argtypes = [vp]
    L.flod_abi_version.restype = C.c_int
    _lib = L
    return L


def camera_struct(cam) -> CameraStruct:
    """Marshal any object with the fields of flod_camera (e.g. flod_synth.Camera)."""
    c = CameraStruct()
    c.R[:] = [float(v) for v in np.asarray(cam.R, dtype=np.float32).reshape(9)]
    c.t[:] = [float(v) for v in np.asarray(cam.t, dtype=np.float32).reshape(3)]
    c.fx, c.fy, c.cx, c.cy = cam.fx, cam.fy, cam.cx, cam.cy
    c.width, c.height, c.z_near = int(cam.width), int(cam.height), cam.z_near
    c.bg[:] = [float(v) for v in cam.bg]
    return c


def _f32(a):
    return np.ascontiguousarray(a, dtype=np.float32)


class Renderer:
    """One flod_ctx plus the torch tensors that back its arena and workspace.  Method names follow the C ABI."""

    def __init__(self, device: int = 0):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2408_12894_b200 needs a CUDA device (no CPU fallback)")
        self._torch = torch
        self.lib = load_library()
        self.device = torch.device("cuda", device)
        torch.cuda.init()
        with torch.cuda.device(self.device):
            torch.empty(1, device=self.device)     # make sure the primary context exists
        h = C.c_void_p()
        rc = self.lib.flod_create(C.byref(h), device)
        if rc:
            raise FlodError(rc, "flod_create failed")
        self._h = h
        self.arena = None
        self.workspace = None
        self.n_total = 0
        self.ws_dims = None
        self.pair_rule = PAIR_RULE_BOX              # the library's default (include/flod.h)

    def close(self):
        if getattr(self, "_h", None):
            self.lib.flod_destroy(self._h)
            self._h = None

    __del__ = close

    def _check(self, rc):
        if rc:
            raise FlodError(rc, self.lib.flod_last_error(self._h).decode())

    def _stream(self):
        return C.c_void_p(self._torch.cuda.current_stream(self.device).cuda_stream)

    # ---- flod_scene_bytes + flod_upload_levels
    def upload_levels(self, levels, sh_degree: int):
        keep = []
        descs = (LevelDesc * len(levels))()
        for i, lv in enumerate(levels):
            arrs = [_f32(lv.mean), _f32(lv.log_scale), _f32(lv.quat), _f32(lv.opacity_logit), _f32(lv.sh)]
            keep.append(arrs)
            descs[i].n, descs[i].level, descs[i].s_min = arrs[0].shape[0], lv.level, lv.s_min
            (descs[i].mean, descs[i].log_scale, descs[i].quat, descs[i].opacity_logit,
             descs[i].sh) = [a.ctypes.data for a in arrs]
        nbytes = self.lib.flod_scene_bytes(len(levels), descs, sh_degree)
        if nbytes == 0:
            raise FlodError(-1, "flod_scene_bytes rejected the level list")
        self.arena = self._torch.empty(nbytes, dtype=self._torch.uint8, device=self.device)
        self._check(self.lib.flod_upload_levels(self._h, len(levels), descs, sh_degree,
                                                C.c_void_p(self.arena.data_ptr()), nbytes, self._stream()))
        self.n_total = sum(a[0].shape[0] for a in keep)
        self.workspace = None
        return nbytes

    # ---- flod_workspace_bytes + flod_set_workspace
    def set_workspace(self, width: int, height: int, max_pairs: int):
        nbytes = self.lib.flod_workspace_bytes(self._h, width, height, max_pairs)
        if nbytes == 0:
            raise FlodError(-1, "flod_workspace_bytes rejected the arguments (or no scene uploaded)")
        self.workspace = self._torch.empty(nbytes, dtype=self._torch.uint8, device=self.device)
        self._check(self.lib.flod_set_workspace(self._h, C.c_void_p(self.workspace.data_ptr()), nbytes,
                                                width, height, max_pairs))
        self.ws_dims = (width, height, max_pairs)
        return nbytes

    def set_selection_reference(self, ref_pos=None):
        if ref_pos is None:
            self._check(self.lib.flod_set_selection_reference(self._h, None))
        else:
            arr = (C.c_float * 3)(*[float(np.float32(v)) for v in ref_pos])
            self._check(self.lib.flod_set_selection_reference(self._h, arr))

    def set_pair_rule(self, rule: int):
        self._check(self.lib.flod_set_pair_rule(self._h, rule))
        self.pair_rule = rule

    def set_options(self, flags: int):
        self._check(self.lib.flod_set_options(self._h, flags))

    # ---- flod_render
    def render(self, cam, l_start: int, l_end: int, gamma: float, out=None):
        cs = cam if isinstance(cam, CameraStruct) else camera_struct(cam)
        if out is None:
            out = self._torch.empty((3, cs.height, cs.width), dtype=self._torch.float32, device=self.device)
        self._check(self.lib.flod_render(self._h, C.byref(cs), LevelMode(l_start, l_end), float(gamma),
                                         C.c_void_p(out.data_ptr()), self._stream()))
        return out

    # ---- flod_render_rows: the strip of tile rows [ty_begin, ty_end) into a [3][rows][W] buffer
    def render_rows(self, cam, l_start: int, l_end: int, gamma: float, ty_begin: int, ty_end: int, out=None):
        cs = cam if isinstance(cam, CameraStruct) else camera_struct(cam)
        rows = max(0, min(cs.height, 16 * ty_end) - 16 * ty_begin)
        if out is None:
            out = self._torch.empty((3, rows, cs.width), dtype=self._torch.float32, device=self.device)
        ptr = out.data_ptr() if out.numel() else self.arena.data_ptr()      # (an empty strip writes nothing; any non-null pointer)
        self._check(self.lib.flod_render_rows(self._h, C.byref(cs), LevelMode(l_start, l_end), float(gamma),
                                              int(ty_begin), int(ty_end), C.c_void_p(ptr), self._stream()))
        return out

    # ---- flod_render_to_host: host buffer in, host buffer out
    def render_to_host(self, cam, l_start: int, l_end: int, gamma: float, out_host=None):
        cs = cam if isinstance(cam, CameraStruct) else camera_struct(cam)
        if out_host is None:
            out_host = self._torch.empty((3, cs.height, cs.width), dtype=self._torch.float32, pin_memory=True)
        self._check(self.lib.flod_render_to_host(self._h, C.byref(cs), LevelMode(l_start, l_end), float(gamma),
                                                 C.c_void_p(out_host.data_ptr()), self._stream()))
        return out_host

    # ---- flod_render_to_host_async / flod_wait_host: kernels on the current stream, copy on `copy_stream`
    def render_to_host_async(self, cam, l_start: int, l_end: int, gamma: float, out_host, copy_stream):
        cs = cam if isinstance(cam, CameraStruct) else camera_struct(cam)
        self._check(self.lib.flod_render_to_host_async(self._h, C.byref(cs), LevelMode(l_start, l_end), float(gamma),
                                                       C.c_void_p(out_host.data_ptr()), self._stream(),
                                                       C.c_void_p(copy_stream.cuda_stream)))
        return out_host

    def wait_host(self):
        self._check(self.lib.flod_wait_host(self._h))

    # ---- materialised G_sel: flod_subset_bytes + flod_subset_set_arena, flod_subset_build / ready / swap, flod_render_subset
    def subset_set_arena(self, l_start: int, l_end: int):
        nbytes = self.lib.flod_subset_bytes(self._h, LevelMode(l_start, l_end))
        if nbytes == 0:
            raise FlodError(-2, "flod_subset_bytes rejected the level range (or no scene uploaded)")
        self.subset_arena = self._torch.empty(nbytes, dtype=self._torch.uint8, device=self.device)
        self._check(self.lib.flod_subset_set_arena(self._h, C.c_void_p(self.subset_arena.data_ptr()), nbytes,
                                                   LevelMode(l_start, l_end)))
        return nbytes

    def subset_build(self, ref_pos, fx: float, gamma: float, stream=None):
        arr = (C.c_float * 3)(*[float(np.float32(v)) for v in ref_pos])
        st = self._stream() if stream is None else C.c_void_p(stream.cuda_stream)
        self._check(self.lib.flod_subset_build(self._h, arr, float(fx), float(gamma), st))

    def subset_ready(self) -> bool:
        rc = self.lib.flod_subset_ready(self._h)
        if rc < 0:
            self._check(rc)
        return rc == 1

    def subset_swap(self) -> int:
        n = C.c_int64(0)
        self._check(self.lib.flod_subset_swap(self._h, C.byref(n)))
        return n.value

    def render_subset(self, cam, out=None):
        cs = cam if isinstance(cam, CameraStruct) else camera_struct(cam)
        if out is None:
            out = self._torch.empty((3, cs.height, cs.width), dtype=self._torch.float32, device=self.device)
        self._check(self.lib.flod_render_subset(self._h, C.byref(cs), C.c_void_p(out.data_ptr()), self._stream()))
        return out

    # ---- flod_render_backward: gradients of <upstream, image> of the last frame rendered by render()
    def render_backward(self, cam, upstream, sh_degree: int):
        """upstream: CUDA float32 [3, H, W].  Returns a dict of CUDA float32 tensors indexed by gid."""
        t = self._torch
        cs = cam if isinstance(cam, CameraStruct) else camera_struct(cam)
        n, K = max(self.n_total, 1), (sh_degree + 1) ** 2
        z = lambda *shape: t.empty(shape, dtype=t.float32, device=self.device)
        out = {"mean": z(n, 3), "log_scale": z(n, 3), "quat": z(n, 4), "logit": z(n), "sh": z(n, K, 3)}
        g = Grads(*[C.c_void_p(out[k].data_ptr()) for k in ("mean", "log_scale", "quat", "logit", "sh")])
        nbytes = self.lib.flod_backward_workspace_bytes(self._h)
        if getattr(self, "bwd_workspace", None) is None or self.bwd_workspace.numel() < nbytes:
            self.bwd_workspace = t.empty(nbytes, dtype=t.uint8, device=self.device)
        upstream = upstream.contiguous()
        self._check(self.lib.flod_render_backward(self._h, C.byref(cs), C.c_void_p(upstream.data_ptr()), C.byref(g),
                                                  C.c_void_p(self.bwd_workspace.data_ptr()), nbytes, self._stream()))
        return {k: v[:self.n_total] for k, v in out.items()}

    def launches_per_frame(self) -> int:
        return self.lib.flod_launches_per_frame(self._h)

    # ---- flod_get_stats
    def get_stats(self, raise_on_overflow: bool = True) -> dict:
        st = Stats()
        rc = self.lib.flod_get_stats(self._h, C.byref(st))
        if rc and (raise_on_overflow or rc != -5):
            self._check(rc)
        d = {k: getattr(st, k) for k in ("n_scan", "n_sel", "n_front", "n_vis", "n_pairs", "max_pairs",
                                         "overflow", "evals", "blends", "ms_total")}
        d["ms_stage"] = list(st.ms_stage)
        return d

    # ---- flod_debug_copy
    def _dbg(self, what, arr):
        self._check(self.lib.flod_debug_copy(self._h, what, C.c_void_p(arr.ctypes.data), arr.nbytes))
        return arr

    def debug_mask(self):
        return self._dbg(FLOD_DBG_MASK, np.zeros(max(self.n_total, 1), np.uint8))[:self.n_total]

    def debug_tile_counts(self, n_tiles: int):
        return self._dbg(FLOD_DBG_TILE_COUNTS, np.zeros(n_tiles, np.uint32))

    def debug_projected(self, n_vis: int):
        return self._dbg(FLOD_DBG_PROJECTED, np.zeros(max(n_vis, 1), DBG_PROJECTED_DTYPE))[:n_vis]

    def debug_sorted_pairs(self, n_pairs: int):
        return self._dbg(FLOD_DBG_SORTED_PAIRS, np.zeros(max(n_pairs, 1), DBG_PAIR_DTYPE))[:n_pairs]

    def debug_activated(self):
        return self._dbg(FLOD_DBG_ACTIVATED, np.zeros((max(self.n_total, 1), 8), np.float32))[:self.n_total]


# ---- flod_overlap_prune (training-side): no context, caller-owned device arrays
def overlap_prune(mean, s_min: float, with_distances: bool = True):
    """mean: CUDA float32 tensor [n, 3].  Returns (remove uint8 [n], mean 3-NN distance float32 [n] or None)."""
    import torch
    if not (mean.is_cuda and mean.dtype == torch.float32 and mean.dim() == 2 and mean.shape[1] == 3):
        raise ValueError("overlap_prune wants a CUDA float32 tensor of shape [n, 3]")
    lib = load_library()
    mean = mean.contiguous()
    n = mean.shape[0]
    remove = torch.zeros(n, dtype=torch.uint8, device=mean.device)
    dist = torch.full((n,), float("inf"), dtype=torch.float32, device=mean.device) if with_distances else None
    if n == 0:
        return remove, dist
    lo = mean.min(dim=0).values.cpu().numpy().astype(np.float32)
    ws = torch.empty(lib.flod_overlap_prune_workspace_bytes(n), dtype=torch.uint8, device=mean.device)
    with torch.cuda.device(mean.device):
        rc = lib.flod_overlap_prune(C.c_void_p(mean.data_ptr()), n, float(s_min), (C.c_float * 3)(*[float(v) for v in lo]),
                                    C.c_void_p(remove.data_ptr()), C.c_void_p(dist.data_ptr()) if dist is not None else None,
                                    C.c_void_p(ws.data_ptr()), ws.numel(),
                                    C.c_void_p(torch.cuda.current_stream(mean.device).cuda_stream))
        torch.cuda.current_stream(mean.device).synchronize()      # the workspace is freed on return
    if rc:
        raise FlodError(rc, "flod_overlap_prune rejected its arguments")
    return remove, dist


def overlap_prune_static_max_n() -> int:
    return int(load_library().flod_overlap_prune_static_max_n())


def overlap_prune_static(mean, s_min: float, bbox_lo, remove, dist=None):
    """flod_overlap_prune_static: overlap_prune without a workspace, for callers that may not allocate device memory.
    The scratch is a fixed array inside the library, so n <= overlap_prune_static_max_n() (FlodError otherwise), and every
    call on a device shares it: calls that overlap on the GPU race.  Nothing is allocated here either: the caller passes
    bbox_lo (three floats <= every mean, componentwise) and the outputs `remove` (uint8 [n]) and `dist` (float32 [n] or
    None), and the call is asynchronous on torch's current stream."""
    import torch
    if not (mean.is_cuda and mean.dtype == torch.float32 and mean.dim() == 2 and mean.shape[1] == 3 and mean.is_contiguous()):
        raise ValueError("overlap_prune_static wants a contiguous CUDA float32 tensor of shape [n, 3]")
    n = mean.shape[0]
    if not (remove.is_cuda and remove.dtype == torch.uint8 and remove.numel() == n and remove.is_contiguous()):
        raise ValueError("remove must be a contiguous CUDA uint8 tensor of n elements")
    if dist is not None and not (dist.is_cuda and dist.dtype == torch.float32 and dist.numel() == n and dist.is_contiguous()):
        raise ValueError("dist must be a contiguous CUDA float32 tensor of n elements")
    lib = load_library()
    with torch.cuda.device(mean.device):
        rc = lib.flod_overlap_prune_static(C.c_void_p(mean.data_ptr()), n, float(s_min), (C.c_float * 3)(*[float(v) for v in bbox_lo]),
                                           C.c_void_p(remove.data_ptr()), C.c_void_p(dist.data_ptr()) if dist is not None else None,
                                           C.c_void_p(torch.cuda.current_stream(mean.device).cuda_stream))
    if rc == -8:
        raise FlodError(rc, f"n = {n} exceeds the built-in scratch (at most {overlap_prune_static_max_n()} points): use overlap_prune")
    if rc:
        raise FlodError(rc, "flod_overlap_prune_static rejected its arguments")
