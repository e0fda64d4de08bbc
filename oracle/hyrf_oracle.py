"""ctypes front-end of the CPU oracle (oracle/hyrf_oracle.c).

TEST INFRASTRUCTURE, NOT PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference legs may import this. It never imports the CUDA binding and shares no code with csrc/.
Scenes come in as objects with the attribute names of `paper_2509_17083_b200.synth.Scene` (duck-typed; the
generator module is not imported here).
"""
from __future__ import annotations

import ctypes as C
import hashlib
import os
import subprocess
from typing import Dict, Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "hyrf_oracle.c")
HO_MAX_LEVELS = 32


class HoGrid(C.Structure):
    _fields_ = [("levels", C.c_uint32), ("feats", C.c_uint32), ("log2_table", C.c_uint32),
                ("res", C.c_uint32 * HO_MAX_LEVELS)]


class HoMlp(C.Structure):
    _fields_ = [("in_dim", C.c_uint32), ("hidden", C.c_uint32), ("n_hidden", C.c_uint32), ("out_dim", C.c_uint32)]


class HoCamera(C.Structure):
    _fields_ = [("R", C.c_float * 9), ("t", C.c_float * 3), ("fx", C.c_float), ("fy", C.c_float),
                ("cx", C.c_float), ("cy", C.c_float)]


class HoScene(C.Structure):
    _fields_ = [("n", C.c_uint32), ("pos", C.c_void_p), ("rgb_logit", C.c_void_p), ("scale_logit", C.c_void_p),
                ("opacity_logit", C.c_void_p), ("aabb_min", C.c_float * 3), ("aabb_max", C.c_float * 3),
                ("geo_grid", HoGrid), ("app_grid", HoGrid), ("bg_grid", HoGrid),
                ("geo_mlp", HoMlp), ("app_mlp", HoMlp), ("bg_mlp", HoMlp),
                ("geo_table", C.c_void_p), ("app_table", C.c_void_p), ("bg_table", C.c_void_p),
                ("geo_w", C.c_void_p), ("app_w", C.c_void_p), ("bg_w", C.c_void_p),
                ("fp16", C.c_int32), ("pe_octaves", C.c_uint32),
                ("cull_tol", C.c_float), ("z_near", C.c_float), ("bg_radius", C.c_float), ("tau_T", C.c_float),
                ("table_u8", C.c_int32), ("geo_q", C.c_void_p), ("app_q", C.c_void_p), ("bg_q", C.c_void_p)]


def _cpu_has_fma() -> bool:
    try:
        with open("/proc/cpuinfo") as f:
            for line in f:
                if line.startswith("flags"):
                    return " fma " in (line + " ")
    except OSError:
        pass
    return False


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (-O2 -ffp-contract=off; -mfma only when this host has FMA, otherwise glibc's
    correctly rounded fmaf is used — results are identical either way). Returns the .so path."""
    with open(_SRC, "rb") as f:
        digest = hashlib.sha1(f.read()).hexdigest()[:12]
    fma = _cpu_has_fma()
    so = os.path.join(_HERE, f"libhyrf_oracle_{digest}_{'fma' if fma else 'nofma'}.so")
    if force or not os.path.exists(so):
        for old in os.listdir(_HERE):
            if old.startswith("libhyrf_oracle_") and old.endswith(".so") and os.path.join(_HERE, old) != so:
                try:
                    os.remove(os.path.join(_HERE, old))
                except OSError:
                    pass
        cmd = ["gcc", "-std=c11", "-O2", "-ffp-contract=off", "-fno-fast-math", "-fopenmp", "-fPIC", "-shared",
               "-Wall", "-Wextra", "-o", so + ".tmp", _SRC, "-lm"]
        if fma:
            cmd.insert(1, "-mfma")
        subprocess.run(cmd, check=True)
        os.replace(so + ".tmp", so)
    return so


_lib: Optional[C.CDLL] = None


def lib() -> C.CDLL:
    global _lib
    if _lib is None:
        # HYRF_ORACLE_SO: a separately built oracle library (e.g. the -fsanitize=address,undefined build the
        # sanitizer pass of profiles/r2_sanitizer.md runs the CPU tests against)
        L = C.CDLL(os.environ.get("HYRF_ORACLE_SO") or build())
        L.ho_half_to_float.restype = C.c_float
        L.ho_half_to_float.argtypes = [C.c_uint16]
        L.ho_float_to_half.restype = C.c_uint16
        L.ho_float_to_half.argtypes = [C.c_float]
        L.ho_softexp.restype = C.c_float
        L.ho_softexp.argtypes = [C.c_float]
        L.ho_sigmoid.restype = C.c_float
        L.ho_sigmoid.argtypes = [C.c_float]
        L.ho_stage_cull.restype = C.c_uint32
        L.ho_grid_layout.restype = C.c_uint64
        L.ho_grid_index.restype = C.c_uint32
        L.ho_grid_index.argtypes = [C.c_void_p, C.c_uint32, C.c_uint32, C.c_uint32, C.c_uint32]
        L.ho_project.restype = C.c_uint32
        L.ho_stage_project.restype = C.c_uint64
        L.ho_stage_bin.restype = C.c_int32
        L.ho_pair_alpha.restype = C.c_float
        L.ho_num_threads.restype = C.c_int32
        L.ho_decode_explicit.restype = C.c_uint32
        _lib = L
    return _lib


def _p(a: np.ndarray):
    return a.ctypes.data_as(C.c_void_p)


def _f32(a, shape=None) -> np.ndarray:
    a = np.ascontiguousarray(np.asarray(a, dtype=np.float32))
    return a if shape is None else a.reshape(shape)


def grid_struct(g) -> HoGrid:
    s = HoGrid()
    s.levels, s.feats, s.log2_table = len(g.level_res), g.feats, g.log2_table
    for i, r in enumerate(g.level_res):
        s.res[i] = int(r)
    return s


def mlp_struct(m) -> HoMlp:
    return HoMlp(m.in_dim, m.hidden, m.n_hidden, m.out_dim)


def camera_struct(cam) -> HoCamera:
    c = HoCamera()
    R = np.asarray(cam.R, dtype=np.float32).reshape(9)
    t = np.asarray(cam.t, dtype=np.float32).reshape(3)
    for i in range(9):
        c.R[i] = float(R[i])
    for i in range(3):
        c.t[i] = float(t[i])
    c.fx, c.fy, c.cx, c.cy = float(cam.fx), float(cam.fy), float(cam.cx), float(cam.cy)
    return c


class OracleScene:
    """Holds the numpy arrays alive and the C struct that points at them."""

    def __init__(self, scene):
        if getattr(scene, "explicit_rvq", None) is not None:   # compressed explicit part: decode it first (D1')
            scene = with_decoded_explicit(scene)
        self.src = scene
        self.fp16 = bool(scene.fp16)
        self.u8 = bool(getattr(scene, "quant8", False))    # 8-bit min-max tables; decoders stay fp16
        if self.u8 and not self.fp16:
            raise ValueError("8-bit tables go with fp16 decoder weights")
        wdt = np.float16 if self.fp16 else np.float32
        tdt = np.uint8 if self.u8 else wdt
        self._keep = dict(
            pos=_f32(scene.pos), rgb=_f32(scene.rgb_logit), sc=_f32(scene.scale_logit), op=_f32(scene.opacity_logit),
            gt=np.ascontiguousarray(scene.geo_table, dtype=tdt), at=np.ascontiguousarray(scene.app_table, dtype=tdt),
            bt=np.ascontiguousarray(scene.bg_table, dtype=tdt), gw=np.ascontiguousarray(scene.geo_w, dtype=wdt),
            aw=np.ascontiguousarray(scene.app_w, dtype=wdt), bw=np.ascontiguousarray(scene.bg_w, dtype=wdt))
        if self.u8:
            self._keep.update(gq=_f32(scene.geo_q), aq=_f32(scene.app_q), bq=_f32(scene.bg_q))
        k = self._keep
        s = HoScene()
        s.n = int(scene.n)
        s.pos, s.rgb_logit, s.scale_logit, s.opacity_logit = (_p(k["pos"]), _p(k["rgb"]), _p(k["sc"]), _p(k["op"]))
        for i in range(3):
            s.aabb_min[i] = float(scene.aabb_min[i])
            s.aabb_max[i] = float(scene.aabb_max[i])
        s.geo_grid, s.app_grid, s.bg_grid = (grid_struct(scene.geo_grid), grid_struct(scene.app_grid),
                                             grid_struct(scene.bg_grid))
        s.geo_mlp, s.app_mlp, s.bg_mlp = (mlp_struct(scene.geo_mlp), mlp_struct(scene.app_mlp),
                                          mlp_struct(scene.bg_mlp))
        s.geo_table, s.app_table, s.bg_table = _p(k["gt"]), _p(k["at"]), _p(k["bt"])
        s.geo_w, s.app_w, s.bg_w = _p(k["gw"]), _p(k["aw"]), _p(k["bw"])
        s.fp16 = int(self.fp16)
        s.pe_octaves = int(scene.dir_pe_octaves)
        s.cull_tol, s.z_near, s.bg_radius, s.tau_T = (float(scene.cull_tol), float(scene.z_near),
                                                      float(scene.bg_radius), float(scene.tau_T))
        s.table_u8 = int(self.u8)
        if self.u8:
            s.geo_q, s.app_q, s.bg_q = _p(k["gq"]), _p(k["aq"]), _p(k["bq"])
        self.c = s
        self.n = int(scene.n)


# ------------------------------------------------------------------------------------------------------------
# scalar / per-item helpers (used by the pin tests)

def softexp(x: float) -> float:
    return float(lib().ho_softexp(C.c_float(x)))


def sigmoid(x: float) -> float:
    return float(lib().ho_sigmoid(C.c_float(x)))


def half_to_float(h: int) -> float:
    return float(lib().ho_half_to_float(C.c_uint16(h)))


def float_to_half(f: float) -> int:
    return int(lib().ho_float_to_half(C.c_float(f)))



def decode_explicit(rvq) -> Dict[str, np.ndarray]:
    """Compressed explicit Gaussians -> the fp32 SoA arrays of a scene (PAPER.md:227-229 items 1-2; DESIGN.md §2 D1').
    `rvq` has the attribute names of synth.ExplicitRVQ: pos_h (3, N) uint16 binary16 bits, codes (S, N) uint16,
    codebooks (S, K, 5) float32 with columns (s_e, alpha_e, c_e[3])."""
    pos_h = np.ascontiguousarray(rvq.pos_h, np.uint16)
    codes = np.ascontiguousarray(rvq.codes, np.uint16)
    books = np.ascontiguousarray(rvq.codebooks, np.float32)
    S, n = codes.shape
    K = books.shape[1]
    assert pos_h.shape == (3, n) and books.shape == (S, K, 5) and S >= 1
    pos = np.zeros((3, n), np.float32)
    sc = np.zeros(n, np.float32)
    op = np.zeros(n, np.float32)
    rgb = np.zeros((3, n), np.float32)
    bad = lib().ho_decode_explicit(C.c_uint32(n), _p(pos_h), C.c_uint32(S), C.c_uint32(K), _p(codes), _p(books),
                                   _p(pos), _p(sc), _p(op), _p(rgb))
    if bad:
        raise ValueError(f"R-VQ code of Gaussian {bad - 1} is outside the codebook (K = {K})")
    return dict(pos=pos, scale_logit=sc, opacity_logit=op, rgb_logit=rgb)


def with_decoded_explicit(scene):
    """A shallow copy of `scene` whose explicit arrays are the decode of scene.explicit_rvq."""
    import copy
    s = copy.copy(scene)
    for k, v in decode_explicit(scene.explicit_rvq).items():
        setattr(s, k, v)
    s.explicit_rvq = None
    return s


def camera_center(cam) -> np.ndarray:
    o = np.zeros(3, np.float32)
    c = camera_struct(cam)
    lib().ho_camera_center(C.byref(c), _p(o))
    return o


def to_camera(cam, p) -> np.ndarray:
    out = np.zeros(3, np.float32)
    c = camera_struct(cam)
    lib().ho_to_camera(C.byref(c), _p(_f32(p)), _p(out))
    return out


def contract(p, amin, amax) -> np.ndarray:
    x = np.zeros(3, np.float32)
    lib().ho_contract(_p(_f32(p)), _p(_f32(amin)), _p(_f32(amax)), _p(x))
    return x


def grid_layout(grid):
    g = grid_struct(grid)
    sizes = np.zeros(g.levels, np.uint32)
    offs = np.zeros(g.levels, np.uint32)
    dense = np.zeros(g.levels, np.uint8)
    total = lib().ho_grid_layout(C.byref(g), _p(sizes), _p(offs), _p(dense))
    return int(total), sizes, offs, dense.astype(bool)


def grid_index(grid, level: int, vx: int, vy: int, vz: int) -> int:
    g = grid_struct(grid)
    return int(lib().ho_grid_index(C.cast(C.byref(g), C.c_void_p), level, vx, vy, vz))


def grid_encode(grid, table: np.ndarray, x, fp16: bool = False, q: Optional[np.ndarray] = None) -> np.ndarray:
    """q given: `table` holds 8-bit codes, q[level][feature] = (min, step)."""
    g = grid_struct(grid)
    feat = np.zeros(g.levels * g.feats, np.float32)
    if q is not None:
        tab = np.ascontiguousarray(table, dtype=np.uint8)
        lib().ho_grid_encode_q(C.byref(g), _p(tab), C.c_int32(2), _p(_f32(q)), _p(_f32(x)), _p(feat))
        return feat
    tab = np.ascontiguousarray(table, dtype=np.float16 if fp16 else np.float32)
    lib().ho_grid_encode(C.byref(g), _p(tab), C.c_int32(int(fp16)), _p(_f32(x)), _p(feat))
    return feat


def view_dir(p, o) -> np.ndarray:
    d = np.zeros(3, np.float32)
    lib().ho_view_dir(_p(_f32(p)), _p(_f32(o)), _p(d))
    return d


def dir_pe(d, octaves: int = 4, fp16: bool = False) -> np.ndarray:
    out = np.zeros(6 * octaves, np.float32)
    lib().ho_dir_pe(_p(_f32(d)), C.c_uint32(octaves), C.c_int32(int(fp16)), _p(out))
    return out


def mlp_forward(mlp, w: np.ndarray, x, fp16: bool = False) -> np.ndarray:
    m = mlp_struct(mlp)
    wv = np.ascontiguousarray(w, dtype=np.float16 if fp16 else np.float32)
    out = np.zeros(m.out_dim, np.float32)
    lib().ho_mlp_forward(C.byref(m), _p(wv), C.c_int32(int(fp16)), _p(_f32(x)), _p(out))
    return out


def aggregate(raw, s_e: float, a_e: float, c_e) -> np.ndarray:
    out = np.zeros(11, np.float32)
    lib().ho_aggregate(_p(_f32(raw)), C.c_float(s_e), C.c_float(a_e), _p(_f32(c_e)), _p(out))
    return out


def project(attrs, pc, cam, W: int, H: int):
    c = camera_struct(cam)
    proj = np.zeros(10, np.float32)
    cov = np.zeros(3, np.float32)
    radius = C.c_float(0)
    rect = np.zeros(4, np.uint32)
    tiles = lib().ho_project(_p(_f32(attrs)), _p(_f32(pc)), C.byref(c), C.c_int32(W), C.c_int32(H), _p(proj),
                             _p(cov), C.byref(radius), _p(rect))
    return dict(proj=proj, cov=cov, radius=float(radius.value), rect=rect, tiles=int(tiles))


def pair_alpha(proj, i: float, j: float):
    sk = C.c_int32(0)
    a = lib().ho_pair_alpha(_p(_f32(proj)), C.c_float(i), C.c_float(j), C.byref(sk))
    return float(a), bool(sk.value)


def ray_sphere(cam, i: float, j: float, radius: float):
    c = camera_struct(cam)
    d = np.zeros(3, np.float32)
    ps = np.zeros(3, np.float32)
    lib().ho_ray_sphere(C.byref(c), C.c_float(i), C.c_float(j), C.c_float(radius), _p(d), _p(ps))
    return d, ps


def background_color(osc: OracleScene, cam, i: float, j: float) -> np.ndarray:
    c = camera_struct(cam)
    cs = np.zeros(3, np.float32)
    lib().ho_background_color(C.byref(osc.c), C.byref(c), C.c_float(i), C.c_float(j), _p(cs))
    return cs


def query_point(osc: OracleScene, p, o) -> np.ndarray:
    raw = np.zeros(11, np.float32)
    lib().ho_query_point(C.byref(osc.c), _p(_f32(p)), _p(_f32(o)), _p(raw))
    return raw


def set_num_threads(n: int) -> None:
    lib().ho_set_num_threads(C.c_int32(n))


def num_threads() -> int:
    return int(lib().ho_num_threads())


# ------------------------------------------------------------------------------------------------------------
# stages and the whole pass

def stage_cull(osc: OracleScene, cam, W: int, H: int):
    c = camera_struct(cam)
    mask = np.zeros(osc.n, np.uint8)
    idx = np.zeros(osc.n, np.uint32)
    V = lib().ho_stage_cull(C.byref(osc.c), C.byref(c), C.c_int32(W), C.c_int32(H), _p(mask), _p(idx))
    return mask, idx[:V].copy()


def stage_query(osc: OracleScene, cam, vis_idx: np.ndarray) -> np.ndarray:
    c = camera_struct(cam)
    V = len(vis_idx)
    raw = np.zeros((V, 11), np.float32)
    idx = np.ascontiguousarray(vis_idx, dtype=np.uint32)
    lib().ho_stage_query(C.byref(osc.c), C.byref(c), C.c_uint32(V), _p(idx), _p(raw))
    return raw


def stage_aggregate(osc: OracleScene, vis_idx: np.ndarray, raw: np.ndarray) -> np.ndarray:
    V = len(vis_idx)
    attrs = np.zeros((V, 11), np.float32)
    idx = np.ascontiguousarray(vis_idx, dtype=np.uint32)
    lib().ho_stage_aggregate(C.byref(osc.c), C.c_uint32(V), _p(idx), _p(_f32(raw)), _p(attrs))
    return attrs


def stage_project(osc: OracleScene, cam, W: int, H: int, vis_idx: np.ndarray, attrs: np.ndarray):
    c = camera_struct(cam)
    V = len(vis_idx)
    idx = np.ascontiguousarray(vis_idx, dtype=np.uint32)
    proj = np.zeros((V, 10), np.float32)
    cov = np.zeros((V, 3), np.float32)
    radius = np.zeros(V, np.float32)
    rect = np.zeros((V, 4), np.uint32)
    tiles = np.zeros(V, np.uint32)
    D = lib().ho_stage_project(C.byref(osc.c), C.byref(c), C.c_int32(W), C.c_int32(H), C.c_uint32(V), _p(idx),
                               _p(_f32(attrs)), _p(proj), _p(cov), _p(radius), _p(rect), _p(tiles))
    return dict(proj=proj, cov=cov, radius=radius, rect=rect, tiles=tiles, D=int(D))


def stage_bin(W: int, H: int, vis_idx: np.ndarray, proj: np.ndarray, rect: np.ndarray, tiles: np.ndarray):
    V = len(vis_idx)
    D = int(tiles.astype(np.uint64).sum())
    gx, gy = (W + 15) // 16, (H + 15) // 16
    idx = np.ascontiguousarray(vis_idx, dtype=np.uint32)
    list_id = np.zeros(D, np.uint32)
    list_rank = np.zeros(D, np.uint32)
    ranges = np.zeros((gx * gy, 2), np.uint32)
    rc = lib().ho_stage_bin(C.c_int32(W), C.c_int32(H), C.c_uint32(V), _p(idx), _p(_f32(proj)),
                            _p(np.ascontiguousarray(rect, dtype=np.uint32)),
                            _p(np.ascontiguousarray(tiles, dtype=np.uint32)), C.c_uint64(D), _p(list_id),
                            _p(list_rank), _p(ranges))
    if rc != 0:
        raise RuntimeError(f"ho_stage_bin failed: {rc}")
    return dict(list_id=list_id, list_rank=list_rank, ranges=ranges, D=D)


def stage_raster(W: int, H: int, proj: np.ndarray, list_rank: np.ndarray, ranges: np.ndarray):
    cfg = np.zeros((H, W, 3), np.float32)
    T = np.zeros((H, W), np.float32)
    wsum = np.zeros((H, W), np.float32)
    m_alpha = np.zeros((H, W), np.float32)
    m_stop = np.zeros((H, W), np.float32)
    n_eval = np.zeros((H, W), np.uint32)
    n_blend = np.zeros((H, W), np.uint32)
    lib().ho_stage_raster(C.c_int32(W), C.c_int32(H), _p(_f32(proj)),
                          _p(np.ascontiguousarray(list_rank, dtype=np.uint32)),
                          _p(np.ascontiguousarray(ranges, dtype=np.uint32)), _p(cfg), _p(T), _p(wsum), _p(m_alpha),
                          _p(m_stop), _p(n_eval), _p(n_blend))
    return dict(cfg=cfg, T=T, wsum=wsum, m_alpha=m_alpha, m_stop=m_stop, n_eval=n_eval, n_blend=n_blend)


def stage_raster_backward(W: int, H: int, proj: np.ndarray, list_rank: np.ndarray, ranges: np.ndarray,
                          g_cfg: np.ndarray, g_T: np.ndarray) -> np.ndarray:
    """D12: gradients of L w.r.t. the projected records (u, v, A, B, C, o, r, g, b), [V][9] float64, given
    g_cfg = dL/dC_fg [H][W][3] and g_T = dL/dT_final [H][W], with D10's decisions frozen."""
    V = len(proj)
    grad = np.zeros((V, 9), np.float64)
    lib().ho_stage_raster_backward(C.c_int32(W), C.c_int32(H), C.c_uint32(V), _p(_f32(proj)),
                                   _p(np.ascontiguousarray(list_rank, dtype=np.uint32)),
                                   _p(np.ascontiguousarray(ranges, dtype=np.uint32)), _p(_f32(g_cfg, (H, W, 3))),
                                   _p(_f32(g_T, (H, W))), _p(grad))
    return grad


def stage_background(osc: OracleScene, cam, W: int, H: int, cfg: np.ndarray, T: np.ndarray):
    c = camera_struct(cam)
    out = np.zeros((H, W, 3), np.float32)
    bg_mask = np.zeros((H, W), np.uint8)
    lib().ho_stage_background(C.byref(osc.c), C.byref(c), C.c_int32(W), C.c_int32(H), _p(_f32(cfg)), _p(_f32(T)),
                              _p(out), _p(bg_mask))
    return out, bg_mask


# Ablation switches of the same pass (PAPER.md:214-223 Table 5, :233-237, :259-261).
#  NO_CULL     "w/o pre-culling": the fields are queried and aggregated for EVERY stored Gaussian (the overhead the
#              paper's 3.9x is about, :261); Gaussians that fail Eq. 9 are dropped at projection instead (their
#              projected record, rectangle and tiles-touched are zero), so the image is the full model's.
#  NO_BG       "w/o background": out = C_fg, nothing is composited.
#  NO_NEURAL   "w/o neural": all decoder outputs are 0 -> isotropic, diffuse, identity-rotation Gaussians (:237, :259).
#  NO_EXPLICIT "w/o explicit": s_e = alpha_e = c_e = 0 in Eq. 7 (the position stays explicit).
# A single shared field (:233) needs no switch: pass the same table for geo and app.
ABL_NO_CULL, ABL_NO_BG, ABL_NO_NEURAL, ABL_NO_EXPLICIT = 1, 2, 4, 8


def _without_explicit(osc: OracleScene) -> OracleScene:
    import copy
    sc = copy.copy(osc.src)
    sc.rgb_logit = np.zeros_like(_f32(osc.src.rgb_logit))
    sc.scale_logit = np.zeros_like(_f32(osc.src.scale_logit))
    sc.opacity_logit = np.zeros_like(_f32(osc.src.opacity_logit))
    return OracleScene(sc)


def render(osc: OracleScene, cam, W: Optional[int] = None, H: Optional[int] = None,
           attrs_override: Optional[np.ndarray] = None, ablation: int = 0) -> Dict[str, np.ndarray]:
    """The whole pass in the paper's order: cull -> query -> aggregate -> project/bin/sort ->
    rasterise -> background. Returns every intermediate. `attrs_override` replaces the stage-3 output (used by
    the hand-off parity test of SURVEY §8c H1 to drive stages 4-6 from given attributes). `ablation`: ABL_* bits."""
    W = int(cam.W if W is None else W)
    H = int(cam.H if H is None else H)
    mask, vis_idx = stage_cull(osc, cam, W, H)
    in_frustum = None
    if ablation & ABL_NO_CULL:
        in_frustum = mask.astype(bool)
        mask = np.ones(osc.n, np.uint8)
        vis_idx = np.arange(osc.n, dtype=np.uint32)
    raw = np.zeros((len(vis_idx), 11), np.float32) if ablation & ABL_NO_NEURAL else stage_query(osc, cam, vis_idx)
    attrs = stage_aggregate(_without_explicit(osc) if ablation & ABL_NO_EXPLICIT else osc, vis_idx, raw)
    if attrs_override is not None:
        attrs = _f32(attrs_override, (len(vis_idx), 11))
    pr = stage_project(osc, cam, W, H, vis_idx, attrs)
    if in_frustum is not None:
        drop = ~in_frustum
        pr["proj"][drop] = 0.0
        pr["cov"][drop] = 0.0
        pr["radius"][drop] = 0.0
        pr["rect"][drop] = 0
        pr["tiles"][drop] = 0
        pr["D"] = int(pr["tiles"].astype(np.uint64).sum())
    bn = stage_bin(W, H, vis_idx, pr["proj"], pr["rect"], pr["tiles"])
    rs = stage_raster(W, H, pr["proj"], bn["list_rank"], bn["ranges"])
    if ablation & ABL_NO_BG:
        out, bg_mask = rs["cfg"].copy(), np.zeros((H, W), np.uint8)
    else:
        out, bg_mask = stage_background(osc, cam, W, H, rs["cfg"], rs["T"])
    res = dict(mask=mask, vis_idx=vis_idx, raw=raw, attrs=attrs, out=out, bg_mask=bg_mask, W=W, H=H)
    res.update(pr)
    res.update(bn)
    res.update(rs)
    return res
