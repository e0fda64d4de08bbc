"""Thin Python binding of the C-ABI in include/hyrf.h (same names, argument marshalling only).

Every step of the render pass runs inside libhyrf.so's CUDA kernels. PyTorch is used for device memory (the
parameter tensors, the output image) and streams (torch's current stream is handed to hyrf_set_stream). There is
no fallback: if the library is missing or no CUDA device exists, calls raise.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Dict, Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libhyrf.so")

HYRF_OK, HYRF_ERR_INVALID_ARG, HYRF_ERR_NOT_READY, HYRF_ERR_UNSUPPORTED, HYRF_ERR_CAMERA, HYRF_ERR_OOM, HYRF_ERR_CUDA = range(7)
STATUS_NAMES = ["HYRF_OK", "HYRF_ERR_INVALID_ARG", "HYRF_ERR_NOT_READY", "HYRF_ERR_UNSUPPORTED", "HYRF_ERR_CAMERA",
                "HYRF_ERR_OOM", "HYRF_ERR_CUDA"]
HYRF_F32, HYRF_F16, HYRF_U8 = 0, 1, 2
HYRF_MLP_AUTO, HYRF_MLP_FMA, HYRF_MLP_MMA, HYRF_MLP_HMMA, HYRF_MLP_WS = 0, 1, 2, 3, 4
(DBG_VIS_MASK, DBG_VIS_IDX, DBG_STAGE2_RAW, DBG_STAGE3_ATTRS, DBG_PROJ, DBG_RECT, DBG_TILE_RANGES, DBG_TILE_LIST,
 DBG_FINAL_T, DBG_BG_MASK, DBG_COUNTERS, DBG_FG) = range(12)
DBG_EXPLICIT = 12   # f32 [8][N]: the explicit parameters as the scene holds them (needs no render, no debug_enable)
DBG_ALL = (1 << 12) - 1

EXPORTS = ["hyrf_create_scene", "hyrf_upload_params", "hyrf_set_stream", "hyrf_render", "hyrf_render_host",
           "hyrf_destroy_scene", "hyrf_last_error", "hyrf_debug_enable", "hyrf_debug_fetch", "hyrf_set_timing",
           "hyrf_stage_times", "hyrf_last_launch_count", "hyrf_set_ablation", "hyrf_render_host_async",
           "hyrf_host_sync", "hyrf_set_sort_overlap", "hyrf_upload_explicit_rvq", "hyrf_last_decode_time", "hyrf_set_raster_mode",
           "hyrf_last_raster_mode", "hyrf_raster_backward", "hyrf_probe_gather", "hyrf_probe_issue", "hyrf_set_pipelining", "hyrf_frame_gap", "hyrf_set_strip", "hyrf_backward", "hyrf_loss_l1_ssim",
           "hyrf_set_retain_lists", "hyrf_loss_l1_ssim_noalloc", "hyrf_set_bin_granularity"]
ABL_NO_CULL, ABL_NO_BG, ABL_NO_NEURAL, ABL_NO_EXPLICIT = 1, 2, 4, 8


class GridDesc(C.Structure):
    _fields_ = [("levels", C.c_uint32), ("feats", C.c_uint32), ("log2_table", C.c_uint32),
                ("level_res", C.POINTER(C.c_uint32))]


class MlpDesc(C.Structure):
    _fields_ = [("in_dim", C.c_uint32), ("hidden", C.c_uint32), ("n_hidden", C.c_uint32), ("out_dim", C.c_uint32)]


ALLOC_FN = C.CFUNCTYPE(C.c_void_p, C.c_size_t, C.c_void_p)
RELEASE_FN = C.CFUNCTYPE(None, C.c_void_p, C.c_void_p)


class SceneDesc(C.Structure):
    _fields_ = [("n_gaussians", C.c_uint32), ("aabb_min", C.c_float * 3), ("aabb_max", C.c_float * 3),
                ("geo_grid", GridDesc), ("app_grid", GridDesc), ("bg_grid", GridDesc),
                ("geo_mlp", MlpDesc), ("app_mlp", MlpDesc), ("bg_mlp", MlpDesc),
                ("dir_pe_octaves", C.c_uint32), ("param_dtype", C.c_int), ("mlp_path", C.c_int),
                ("cull_tol", C.c_float), ("z_near", C.c_float), ("bg_radius", C.c_float), ("tau_T", C.c_float),
                ("max_width", C.c_uint32), ("max_height", C.c_uint32), ("device", C.c_int32),
                ("alloc", ALLOC_FN), ("release", RELEASE_FN), ("user", C.c_void_p)]


class Params(C.Structure):
    _fields_ = [("pos", C.c_void_p), ("rgb_logit", C.c_void_p), ("scale_logit", C.c_void_p),
                ("opacity_logit", C.c_void_p), ("geo_table", C.c_void_p), ("app_table", C.c_void_p),
                ("bg_table", C.c_void_p), ("geo_w", C.c_void_p), ("app_w", C.c_void_p), ("bg_w", C.c_void_p),
                ("geo_q", C.c_void_p), ("app_q", C.c_void_p), ("bg_q", C.c_void_p),
                ("host_ptrs", C.c_int32)]


class ExplicitRvqC(C.Structure):
    _fields_ = [("pos_h", C.c_void_p), ("stages", C.c_uint32), ("codebook_size", C.c_uint32), ("codes", C.c_void_p),
                ("codebooks", C.c_void_p), ("host_ptrs", C.c_int32)]


class GradsC(C.Structure):
    _fields_ = [(n, C.c_void_p) for n in ("pos", "rgb_logit", "scale_logit", "opacity_logit", "geo_table", "app_table",
                                          "bg_table", "geo_w", "app_w", "bg_w")]


class CameraC(C.Structure):
    _fields_ = [("R", C.c_float * 9), ("t", C.c_float * 3), ("fx", C.c_float), ("fy", C.c_float),
                ("cx", C.c_float), ("cy", C.c_float)]


class HyrfError(RuntimeError):
    def __init__(self, status: int, msg: str):
        super().__init__(f"{STATUS_NAMES[status] if 0 <= status < len(STATUS_NAMES) else status}: {msg}")
        self.status = status


_lib: Optional[C.CDLL] = None


def load_library() -> C.CDLL:
    """Load libhyrf.so (built by paper_2509_17083_b200.build). Raises if it is missing: there is no fallback."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise FileNotFoundError(f"{LIB_PATH} not found: run `python -m paper_2509_17083_b200.build` "
                                    "(the CUDA extension is the only implementation; there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        vp = C.c_void_p
        L.hyrf_create_scene.argtypes = [C.POINTER(SceneDesc), C.POINTER(vp)]
        L.hyrf_upload_params.argtypes = [vp, C.POINTER(Params)]
        L.hyrf_set_stream.argtypes = [vp, vp]
        L.hyrf_render.argtypes = [vp, C.POINTER(CameraC), C.c_int32, C.c_int32, vp]
        L.hyrf_render_host.argtypes = [vp, C.POINTER(CameraC), C.c_int32, C.c_int32, vp]
        L.hyrf_destroy_scene.argtypes = [vp]
        L.hyrf_last_error.restype = C.c_char_p
        L.hyrf_debug_enable.argtypes = [vp, C.c_uint32]
        L.hyrf_debug_fetch.argtypes = [vp, C.c_uint32, vp, C.c_size_t, C.POINTER(C.c_size_t)]
        L.hyrf_set_timing.argtypes = [vp, C.c_int32]
        L.hyrf_stage_times.argtypes = [vp, C.POINTER(C.c_float)]
        L.hyrf_last_launch_count.argtypes = [vp, C.POINTER(C.c_uint32)]
        L.hyrf_set_ablation.argtypes = [vp, C.c_uint32]
        L.hyrf_set_sort_overlap.argtypes = [vp, C.c_int]
        L.hyrf_set_pipelining.argtypes = [vp, C.c_int]
        L.hyrf_frame_gap.argtypes = [vp, C.POINTER(C.c_float)]
        L.hyrf_set_strip.argtypes = [vp, C.c_int32, C.c_int32]
        L.hyrf_backward.argtypes = [vp, vp, C.POINTER(GradsC)]
        L.hyrf_loss_l1_ssim.argtypes = [vp, vp, vp, C.c_int32, C.c_int32, C.c_float, C.POINTER(C.c_double), vp]
        L.hyrf_render_host_async.argtypes = [vp, C.POINTER(CameraC), C.c_int32, C.c_int32, vp]
        L.hyrf_host_sync.argtypes = [vp]
        L.hyrf_upload_explicit_rvq.argtypes = [vp, C.POINTER(ExplicitRvqC)]
        L.hyrf_last_decode_time.argtypes = [vp, C.POINTER(C.c_float)]
        L.hyrf_set_raster_mode.argtypes = [vp, C.c_int]
        L.hyrf_last_raster_mode.argtypes = [vp, C.POINTER(C.c_int)]
        L.hyrf_raster_backward.argtypes = [vp, vp, vp, vp, C.c_uint64]
        L.hyrf_set_retain_lists.argtypes = [vp, C.c_int]
        L.hyrf_set_bin_granularity.argtypes = [vp, C.c_int]
        L.hyrf_loss_l1_ssim_noalloc.argtypes = [C.c_int32, vp, vp, vp, C.c_int32, C.c_int32, C.c_float, C.POINTER(C.c_double), vp]
        L.hyrf_probe_gather.argtypes = [C.c_int32, C.c_uint64, C.c_uint32, C.c_uint32, C.c_uint32, C.c_uint32, C.c_uint32,
                                        C.POINTER(C.c_double), C.POINTER(C.c_double), C.POINTER(C.c_float)]
        L.hyrf_probe_issue.argtypes = [C.c_int32, C.c_uint32, C.c_uint32, C.c_uint32, C.POINTER(C.c_double),
                                       C.POINTER(C.c_float)]
        for name in EXPORTS:
            if name != "hyrf_last_error":
                getattr(L, name).restype = C.c_int
        _lib = L
    return _lib


def last_error() -> str:
    return load_library().hyrf_last_error().decode(errors="replace")


def _check(status: int) -> None:
    if status != HYRF_OK:
        raise HyrfError(status, last_error())


LOSS_NOALLOC_MAX_PIXELS = 1 << 20   # include/hyrf.h HYRF_LOSS_NOALLOC_MAX_PIXELS


def loss_l1_ssim_noalloc(image, target, lam: float = 0.2, g_image=None):
    """hyrf_loss_l1_ssim_noalloc (include/hyrf.h): the Eq. 12 loss without any allocation by the library. image, target:
    (H, W, 3) float32 contiguous CUDA tensors; g_image: a caller-owned tensor of the same shape that receives
    dL/d image, or None. Runs on torch's current stream of the tensors' device. Returns the loss."""
    import torch
    if not (image.is_contiguous() and target.is_contiguous() and (g_image is None or g_image.is_contiguous())):
        raise ValueError("loss_l1_ssim_noalloc: contiguous tensors only (making a copy would allocate)")
    H, W = int(image.shape[0]), int(image.shape[1])
    dev = image.device.index if image.device.index is not None else torch.cuda.current_device()
    loss = C.c_double(0)
    _check(load_library().hyrf_loss_l1_ssim_noalloc(
        dev, C.c_void_p(torch.cuda.current_stream(dev).cuda_stream), C.c_void_p(image.data_ptr()),
        C.c_void_p(target.data_ptr()), W, H, C.c_float(lam), C.byref(loss),
        C.c_void_p(g_image.data_ptr() if g_image is not None else None)))
    return float(loss.value)


def probe_gather(device: int, table_bytes: int, entry_bytes: int, ctas_per_sm: int, share: int = 1, line: int = 0,
                 iters: int = 256):
    """hyrf_probe_gather (include/hyrf.h): (lane look-ups per second, distinct sectors per second, ms)."""
    a, b, ms = C.c_double(0), C.c_double(0), C.c_float(0)
    _check(load_library().hyrf_probe_gather(device, table_bytes, entry_bytes, ctas_per_sm, share, line, iters,
                                            C.byref(a), C.byref(b), C.byref(ms)))
    return float(a.value), float(b.value), float(ms.value)


def probe_issue(device: int, kind: int, ctas_per_sm: int, iters: int = 4096):
    """hyrf_probe_issue (include/hyrf.h): (warp instructions per second, ms)."""
    a, ms = C.c_double(0), C.c_float(0)
    _check(load_library().hyrf_probe_issue(device, kind, ctas_per_sm, iters, C.byref(a), C.byref(ms)))
    return float(a.value), float(ms.value)


def camera_struct(cam) -> CameraC:
    c = CameraC()
    R = np.asarray(cam.R, dtype=np.float32).reshape(9)
    t = np.asarray(cam.t, dtype=np.float32).reshape(3)
    for i in range(9):
        c.R[i] = float(R[i])
    for i in range(3):
        c.t[i] = float(t[i])
    c.fx, c.fy, c.cx, c.cy = float(cam.fx), float(cam.fy), float(cam.cx), float(cam.cy)
    return c


def _grid_desc(g, keep: list) -> GridDesc:
    arr = (C.c_uint32 * len(g.level_res))(*[int(r) for r in g.level_res])
    keep.append(arr)
    return GridDesc(len(g.level_res), int(g.feats), int(g.log2_table), C.cast(arr, C.POINTER(C.c_uint32)))


def make_desc(scene, max_width: int, max_height: int, device: int = 0, mlp_path: int = HYRF_MLP_AUTO,
              keep: Optional[list] = None, allocator=None) -> SceneDesc:
    """hyrf_scene_desc from an object with the attribute names of synth.Scene. `allocator`: optional object with
    alloc(nbytes) -> device address (0 on failure) and release(address); it becomes hyrf_scene_desc.alloc / .release."""
    keep = keep if keep is not None else []
    d = SceneDesc()
    d.n_gaussians = int(scene.n)
    for i in range(3):
        d.aabb_min[i] = float(scene.aabb_min[i])
        d.aabb_max[i] = float(scene.aabb_max[i])
    d.geo_grid, d.app_grid, d.bg_grid = (_grid_desc(scene.geo_grid, keep), _grid_desc(scene.app_grid, keep),
                                         _grid_desc(scene.bg_grid, keep))
    for name in ("geo_mlp", "app_mlp", "bg_mlp"):
        m = getattr(scene, name)
        setattr(d, name, MlpDesc(m.in_dim, m.hidden, m.n_hidden, m.out_dim))
    d.dir_pe_octaves = int(scene.dir_pe_octaves)
    d.param_dtype = HYRF_U8 if getattr(scene, "quant8", False) else (HYRF_F16 if scene.fp16 else HYRF_F32)
    d.mlp_path = int(mlp_path)
    d.cull_tol, d.z_near, d.bg_radius, d.tau_T = (float(scene.cull_tol), float(scene.z_near),
                                                  float(scene.bg_radius), float(scene.tau_T))
    d.max_width, d.max_height, d.device = int(max_width), int(max_height), int(device)
    if allocator is None:
        d.alloc = ALLOC_FN()
        d.release = RELEASE_FN()
    else:
        d.alloc = ALLOC_FN(lambda nbytes, user: allocator.alloc(int(nbytes)) or None)
        d.release = RELEASE_FN(lambda ptr, user: allocator.release(int(ptr or 0)))
        keep.extend([d.alloc, d.release, allocator])
    d.user = None
    d._keep = keep
    return d


_DBG_DTYPE = {DBG_VIS_MASK: np.uint8, DBG_VIS_IDX: np.uint32, DBG_STAGE2_RAW: np.float32,
              DBG_STAGE3_ATTRS: np.float32, DBG_PROJ: np.float32, DBG_RECT: np.uint32, DBG_TILE_RANGES: np.uint32,
              DBG_TILE_LIST: np.uint32, DBG_FINAL_T: np.float32, DBG_BG_MASK: np.uint8, DBG_COUNTERS: np.uint64,
              DBG_FG: np.float32, DBG_EXPLICIT: np.float32}
_DBG_COLS = {DBG_STAGE2_RAW: 11, DBG_STAGE3_ATTRS: 11, DBG_PROJ: 10, DBG_RECT: 4, DBG_TILE_RANGES: 2}


class HyrfScene:
    """hyrf_scene handle. `scene` has synth.Scene's attribute names; parameters are uploaded from torch CUDA
    tensors (device pointers) unless `host_upload=True` (numpy host pointers)."""

    def __init__(self, scene, max_width: Optional[int] = None, max_height: Optional[int] = None, device: int = 0,
                 mlp_path: int = HYRF_MLP_AUTO, host_upload: bool = False, allocator=None):
        import torch
        self._torch = torch
        self.lib = load_library()
        self.device = device
        cams = getattr(scene, "cameras", [])
        mw = max_width or max([c.W for c in cams] + [16])
        mh = max_height or max([c.H for c in cams] + [16])
        self._keep: list = []
        self.desc = make_desc(scene, mw, mh, device, mlp_path, self._keep, allocator)
        self.handle = C.c_void_p()
        _check(self.lib.hyrf_create_scene(C.byref(self.desc), C.byref(self.handle)))
        self.fp16 = bool(scene.fp16)
        self.n = int(scene.n)
        n_w = lambda m: sum(o * i for o, i in m.layer_shapes())
        self._scene_shapes = dict(pos=(3, self.n), rgb_logit=(3, self.n), scale_logit=(self.n,), opacity_logit=(self.n,),
                                  geo_table=(scene.geo_grid.n_entries(), 2), app_table=(scene.app_grid.n_entries(), 2),
                                  bg_table=(scene.bg_grid.n_entries(), 2), geo_w=(n_w(scene.geo_mlp),),
                                  app_w=(n_w(scene.app_mlp),), bg_w=(n_w(scene.bg_mlp),))
        self.upload(scene, host_upload)

    # -- hyrf_upload_params -------------------------------------------------------------------------------
    def upload(self, scene, host_upload: bool = False) -> None:
        torch = self._torch
        wdt = np.float16 if self.fp16 else np.float32
        u8 = bool(getattr(scene, "quant8", False))
        tdt = np.uint8 if u8 else wdt                  # HYRF_U8: 8-bit codes + (min, step) per level and feature
        rvq = getattr(scene, "explicit_rvq", None)     # compressed explicit part: goes through hyrf_upload_explicit_rvq
        host = {} if rvq is not None else dict(
                    pos=np.ascontiguousarray(scene.pos, np.float32), rgb_logit=np.ascontiguousarray(scene.rgb_logit, np.float32),
                    scale_logit=np.ascontiguousarray(scene.scale_logit, np.float32),
                    opacity_logit=np.ascontiguousarray(scene.opacity_logit, np.float32))
        host.update(geo_table=np.ascontiguousarray(scene.geo_table, tdt), app_table=np.ascontiguousarray(scene.app_table, tdt),
                    bg_table=np.ascontiguousarray(scene.bg_table, tdt), geo_w=np.ascontiguousarray(scene.geo_w, wdt),
                    app_w=np.ascontiguousarray(scene.app_w, wdt), bg_w=np.ascontiguousarray(scene.bg_w, wdt))
        if u8:
            host.update(geo_q=np.ascontiguousarray(scene.geo_q, np.float32), app_q=np.ascontiguousarray(scene.app_q, np.float32),
                        bg_q=np.ascontiguousarray(scene.bg_q, np.float32))
        p = Params()
        if host_upload:
            for k, a in host.items():
                setattr(p, k, a.ctypes.data)
            p.host_ptrs = 1
            hold = host
        else:
            dev = {k: torch.from_numpy(a).to(f"cuda:{self.device}") for k, a in host.items()}
            torch.cuda.synchronize(self.device)
            for k, tns in dev.items():
                setattr(p, k, tns.data_ptr())
            p.host_ptrs = 0
            hold = dev
        self.set_stream()
        _check(self.lib.hyrf_upload_params(self.handle, C.byref(p)))
        del hold
        if rvq is not None:
            self.upload_explicit_rvq(rvq, host_upload)

    # -- hyrf_upload_explicit_rvq ---------------------------------------------------------------------------
    def upload_explicit_rvq(self, rvq, host_upload: bool = False) -> None:
        """rvq has synth.ExplicitRVQ's attribute names: pos_h (3, N) uint16, codes (S, N) uint16, codebooks (S, K, 5)."""
        torch = self._torch
        codes = np.ascontiguousarray(rvq.codes, np.uint16)
        books = np.ascontiguousarray(rvq.codebooks, np.float32)
        pos_h = np.ascontiguousarray(rvq.pos_h, np.uint16)
        if pos_h.shape != (3, self.n) or codes.ndim != 2 or codes.shape[1] != self.n or books.shape != (codes.shape[0], books.shape[1], 5):
            raise ValueError("explicit_rvq arrays do not have the shapes (3, N), (S, N), (S, K, 5)")
        q = ExplicitRvqC()
        q.stages, q.codebook_size = int(codes.shape[0]), int(books.shape[1])
        if host_upload:
            hold = (pos_h, codes, books)
            q.pos_h, q.codes, q.codebooks, q.host_ptrs = pos_h.ctypes.data, codes.ctypes.data, books.ctypes.data, 1
        else:
            # torch has no uint16 arithmetic but carries the bytes: view as int16
            hold = tuple(torch.from_numpy(a.view(np.int16) if a.dtype == np.uint16 else a).to(f"cuda:{self.device}")
                         for a in (pos_h, codes, books))
            torch.cuda.synchronize(self.device)
            q.pos_h, q.codes, q.codebooks, q.host_ptrs = hold[0].data_ptr(), hold[1].data_ptr(), hold[2].data_ptr(), 0
        self.set_stream()
        _check(self.lib.hyrf_upload_explicit_rvq(self.handle, C.byref(q)))
        del hold

    def last_decode_time(self) -> float:
        ms = C.c_float(0)
        _check(self.lib.hyrf_last_decode_time(self.handle, C.byref(ms)))
        return float(ms.value)

    def explicit_params(self) -> np.ndarray:
        """(8, N) float32: p_e[3], s_e, alpha_e, c_e[3] as the scene holds them (HYRF_DBG_EXPLICIT)."""
        return self.debug_fetch(DBG_EXPLICIT).reshape(8, self.n)

    def set_stream(self, stream=None) -> None:
        torch = self._torch
        st = stream if stream is not None else torch.cuda.current_stream(self.device)
        _check(self.lib.hyrf_set_stream(self.handle, C.c_void_p(st.cuda_stream)))

    # -- hyrf_render / hyrf_render_host --------------------------------------------------------------------
    def render(self, cam, W: Optional[int] = None, H: Optional[int] = None, out=None):
        torch = self._torch
        W = int(cam.W if W is None else W)
        H = int(cam.H if H is None else H)
        if out is None:
            out = torch.empty((H, W, 3), dtype=torch.float32, device=f"cuda:{self.device}")
        c = camera_struct(cam)
        self.set_stream()   # torch's current stream may have changed since the upload (`out` was allocated on it)
        _check(self.lib.hyrf_render(self.handle, C.byref(c), W, H, C.c_void_p(out.data_ptr())))
        return out

    def render_struct(self, cam_struct: CameraC, W: int, H: int, out_ptr: int) -> None:
        """The bare call (what bench.py times): the scene keeps the stream of the last set_stream()."""
        _check(self.lib.hyrf_render(self.handle, C.byref(cam_struct), W, H, C.c_void_p(out_ptr)))

    def render_host(self, cam, W: Optional[int] = None, H: Optional[int] = None, out=None):
        torch = self._torch
        W = int(cam.W if W is None else W)
        H = int(cam.H if H is None else H)
        if out is None:
            out = torch.empty((H, W, 3), dtype=torch.float32).pin_memory()
        c = camera_struct(cam)
        _check(self.lib.hyrf_render_host(self.handle, C.byref(c), W, H, C.c_void_p(out.data_ptr())))
        return out

    def render_host_async(self, cam_struct: CameraC, W: int, H: int, out) -> None:
        """Pipelined delivery (hyrf_render_host_async): `out` is a pinned host tensor; alternate between two of them
        and call host_sync() before reading."""
        _check(self.lib.hyrf_render_host_async(self.handle, C.byref(cam_struct), W, H, C.c_void_p(out.data_ptr())))

    def host_sync(self) -> None:
        _check(self.lib.hyrf_host_sync(self.handle))

    # -- debug / measurement --------------------------------------------------------------------------------
    def debug_enable(self, mask: int = DBG_ALL) -> None:
        _check(self.lib.hyrf_debug_enable(self.handle, C.c_uint32(mask)))

    def debug_fetch(self, kind: int) -> np.ndarray:
        need = C.c_size_t(0)
        _check(self.lib.hyrf_debug_fetch(self.handle, kind, None, 0, C.byref(need)))
        dt = np.dtype(_DBG_DTYPE[kind])
        buf = np.zeros(max(need.value // dt.itemsize, 0), dtype=dt)
        if need.value:
            _check(self.lib.hyrf_debug_fetch(self.handle, kind, buf.ctypes.data, buf.nbytes, C.byref(need)))
        cols = _DBG_COLS.get(kind)
        return buf.reshape(-1, cols) if cols else buf

    def debug_all(self, W: int, H: int) -> Dict[str, np.ndarray]:
        f = self.debug_fetch
        return dict(mask=f(DBG_VIS_MASK), vis_idx=f(DBG_VIS_IDX), raw=f(DBG_STAGE2_RAW), attrs=f(DBG_STAGE3_ATTRS),
                    proj=f(DBG_PROJ), rect=f(DBG_RECT), ranges=f(DBG_TILE_RANGES), list_id=f(DBG_TILE_LIST),
                    T=f(DBG_FINAL_T).reshape(H, W), bg_mask=f(DBG_BG_MASK).reshape(H, W), counters=f(DBG_COUNTERS),
                    cfg=f(DBG_FG).reshape(H, W, 3))

    def set_ablation(self, mask: int) -> None:
        """Ablation switches of include/hyrf.h (Table 5): ABL_NO_CULL | ABL_NO_BG | ABL_NO_NEURAL | ABL_NO_EXPLICIT."""
        _check(self.lib.hyrf_set_ablation(self.handle, int(mask)))

    def set_sort_overlap(self, on: bool = True) -> None:
        """Depth sort beside the field query on a second stream (default) or the whole frame serialised (include/hyrf.h)."""
        _check(self.lib.hyrf_set_sort_overlap(self.handle, int(on)))   # (an int > 1: SMs left to the sort, include/hyrf.h)

    def set_strip(self, row_begin: int = 0, row_end: int = 0) -> None:
        """Screen strips over several devices (include/hyrf.h hyrf_set_strip); (0, 0) = the whole image."""
        _check(self.lib.hyrf_set_strip(self.handle, int(row_begin), int(row_end)))

    def set_pipelining(self, on: bool = True) -> None:
        """A stream of hyrf_render calls: frame k+1's cull and depth sort beside frame k's rasterizer (include/hyrf.h)."""
        _check(self.lib.hyrf_set_pipelining(self.handle, int(on)))

    def set_bin_granularity(self, shift: int = 0) -> None:
        """Macro tiles of 2^shift x 2^shift tiles for the binning (0: chosen per frame; include/hyrf.h); same bits, different cost."""
        _check(self.lib.hyrf_set_bin_granularity(self.handle, int(shift)))

    def set_retain_lists(self, on: bool = True) -> None:
        """Training mode: every render keeps the per-tile lists the backward entry points need (include/hyrf.h)."""
        _check(self.lib.hyrf_set_retain_lists(self.handle, int(on)))

    def set_raster_mode(self, mode: int = 0) -> None:
        """0 auto, 1 a pixel per thread, 2 per-warp lists, 3 per-warp lists with two pixels per lane, 4 two pixels per lane over every
        entry (include/hyrf.h hyrf_set_raster_mode); same bits, different cost."""
        _check(self.lib.hyrf_set_raster_mode(self.handle, int(mode)))

    def raster_backward(self, g_cfg, g_T, n_visible: int):
        """hyrf_raster_backward: g_cfg (H, W, 3) and g_T (H, W) float32 CUDA tensors -> (V, 9) float32 CUDA tensor."""
        torch = self._torch
        grad = torch.empty((int(n_visible), 9), dtype=torch.float32, device=f"cuda:{self.device}")
        g_cfg, g_T = g_cfg.contiguous(), g_T.contiguous()
        self.set_stream()
        _check(self.lib.hyrf_raster_backward(self.handle, C.c_void_p(g_cfg.data_ptr()), C.c_void_p(g_T.data_ptr()),
                                             C.c_void_p(grad.data_ptr()), C.c_uint64(grad.shape[0])))
        return grad

    def backward(self, g_out, grads: Optional[Dict] = None, want=None) -> Dict:
        """hyrf_backward: g_out (H, W, 3) float32 CUDA tensor = dL/d out of the last rendered frame -> dict of float32 CUDA
        tensors shaped like the parameters (gradients are ADDED into `grads` when given, else into fresh zeros).
        `want`: names to compute (default all)."""
        torch = self._torch
        sc = self._scene_shapes
        names = list(sc) if want is None else list(want)
        if grads is None:
            grads = {k: torch.zeros(sc[k], dtype=torch.float32, device=f"cuda:{self.device}") for k in names}
        g = GradsC()
        for k in names:
            setattr(g, k, grads[k].data_ptr())
        g_out = g_out.contiguous()
        self.set_stream()
        _check(self.lib.hyrf_backward(self.handle, C.c_void_p(g_out.data_ptr()), C.byref(g)))
        return grads

    def loss_l1_ssim(self, image, target, lam: float = 0.2, want_grad: bool = True):
        """hyrf_loss_l1_ssim (Eq. 12): (H, W, 3) float32 CUDA tensors -> (L, dL/d image or None)."""
        torch = self._torch
        image, target = image.contiguous(), target.contiguous()
        H, W = int(image.shape[0]), int(image.shape[1])
        g = torch.empty_like(image) if want_grad else None
        loss = C.c_double(0)
        self.set_stream()
        _check(self.lib.hyrf_loss_l1_ssim(self.handle, C.c_void_p(image.data_ptr()), C.c_void_p(target.data_ptr()), W, H,
                                          C.c_float(lam), C.byref(loss), C.c_void_p(g.data_ptr() if want_grad else None)))
        return float(loss.value), g

    def last_raster_mode(self) -> int:
        m = C.c_int(0)
        _check(self.lib.hyrf_last_raster_mode(self.handle, C.byref(m)))
        return int(m.value)

    def set_timing(self, on: bool = True) -> None:
        _check(self.lib.hyrf_set_timing(self.handle, int(on)))

    def stage_times(self) -> np.ndarray:
        ms = (C.c_float * 6)()
        _check(self.lib.hyrf_stage_times(self.handle, ms))
        return np.array(list(ms), dtype=np.float64)

    def frame_gap(self) -> float:
        ms = C.c_float(0)
        _check(self.lib.hyrf_frame_gap(self.handle, C.byref(ms)))
        return float(ms.value)

    def last_launch_count(self) -> int:
        n = C.c_uint32(0)
        _check(self.lib.hyrf_last_launch_count(self.handle, C.byref(n)))
        return int(n.value)

    def close(self) -> None:
        if self.handle:
            self.lib.hyrf_destroy_scene(self.handle)
            self.handle = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
