"""Seeded synthetic scenes and cameras for the five BASELINE.json configs (recipe: SURVEY.md §8(d)).

This module is the ONE piece shared by the CPU oracle tests and the CUDA path: it only draws random inputs
(numpy PCG64) and builds camera matrices by the look-at rule. It holds none of the method's arithmetic
(no contraction, hashing, MLP, projection, blending) and imports neither `oracle/` nor the CUDA binding.

The scenes stand in for the paper's trained Mip-NeRF360 / Tanks&Temples / Deep Blending models
(Table 9 :412), which are not available; shapes and sizes follow them.
"""
from __future__ import annotations

import dataclasses
import math
from typing import Dict, List, Optional

import numpy as np

RES_8 = [16, 23, 35, 52, 78, 115, 172, 256]                       # cfg 1 geo/app grids
RES_16 = [16, 22, 30, 42, 58, 80, 111, 153, 212, 294, 406, 561, 776, 1072, 1482, 2048]  # cfg 2-5 geo/app
RES_BG4 = [16, 40, 101, 256]                                      # cfg 1 background grid
RES_BG8 = [16, 32, 64, 128, 256, 512, 1024, 2048]                 # cfg 2-5 background grid (x2.0 growth)
PE_DIMS = 24                                                      # 4 octaves x (sin, cos) x 3 axes


@dataclasses.dataclass
class GridSpec:
    level_res: List[int]
    log2_table: int
    feats: int = 2

    @property
    def levels(self) -> int:
        return len(self.level_res)

    def level_sizes(self) -> List[int]:
        """Entries per level: dense levels (N+1)^3 rounded up to a multiple of 8, hashed levels 2^log2_table.
        (Storage bookkeeping only: needed to know how many random table entries to draw.)"""
        T = 1 << self.log2_table
        out = []
        for n in self.level_res:
            dense = (n + 1) ** 3
            out.append(((dense + 7) // 8) * 8 if dense <= T else T)
        return out

    def n_entries(self) -> int:
        return sum(self.level_sizes())


@dataclasses.dataclass
class MlpSpec:
    in_dim: int
    hidden: int
    n_hidden: int
    out_dim: int

    def layer_shapes(self):
        dims = [self.in_dim] + [self.hidden] * self.n_hidden + [self.out_dim]
        return [(dims[i + 1], dims[i]) for i in range(len(dims) - 1)]

    def n_weights(self) -> int:
        return sum(o * i for o, i in self.layer_shapes())


@dataclasses.dataclass
class Camera:
    R: np.ndarray      # (3,3) float32 row-major world->camera, rows = (right, down, forward)
    t: np.ndarray      # (3,) float32
    fx: float
    fy: float
    cx: float
    cy: float
    W: int
    H: int


@dataclasses.dataclass
class ExplicitRVQ:
    """Compressed explicit Gaussians (PAPER.md:227-229 items 1-2): half-precision positions and residual-VQ codes of
    the five explicit properties. Layout = include/hyrf.h hyrf_explicit_rvq."""
    pos_h: np.ndarray      # (3, N) uint16: IEEE binary16 bit patterns of p_e, SoA
    codes: np.ndarray      # (S, N) uint16: codebook row per stage
    codebooks: np.ndarray  # (S, K, 5) float32: columns (s_e, alpha_e, c_e[0], c_e[1], c_e[2])

    @property
    def stages(self) -> int:
        return int(self.codes.shape[0])

    @property
    def codebook_size(self) -> int:
        return int(self.codebooks.shape[1])

    def nbytes(self) -> int:
        return int(self.pos_h.nbytes + self.codes.nbytes + self.codebooks.nbytes)


@dataclasses.dataclass
class Scene:
    name: str
    n: int
    pos: np.ndarray            # (3, N) float32 SoA
    rgb_logit: np.ndarray      # (3, N) float32
    scale_logit: np.ndarray    # (N,) float32
    opacity_logit: np.ndarray  # (N,) float32
    aabb_min: np.ndarray       # (3,) float32
    aabb_max: np.ndarray       # (3,) float32
    geo_grid: GridSpec
    app_grid: GridSpec
    bg_grid: GridSpec
    geo_mlp: MlpSpec
    app_mlp: MlpSpec
    bg_mlp: MlpSpec
    geo_table: np.ndarray      # (entries, 2) float32 or float16
    app_table: np.ndarray
    bg_table: np.ndarray
    geo_w: np.ndarray          # flat, layers concatenated, each row-major [out][in]
    app_w: np.ndarray
    bg_w: np.ndarray
    fp16: bool
    cull_tol: float = 0.1
    z_near: float = 0.2
    bg_radius: float = 100.0
    tau_T: float = 0.2
    dir_pe_octaves: int = 4
    cameras: List[Camera] = dataclasses.field(default_factory=list)
    # compressed model: tables as 8-bit min-max codes, (entries, 2) uint8, with
    # q[level][feature] = (min, step); decoder weights stay fp16
    quant8: bool = False
    geo_q: Optional[np.ndarray] = None
    app_q: Optional[np.ndarray] = None
    bg_q: Optional[np.ndarray] = None
    # compressed explicit part (PAPER.md:227-229 items 1-2); when set, pos / *_logit above are NOT what is rendered:
    # both sides decode explicit_rvq (the library in hyrf_upload_explicit_rvq, the oracle in decode_explicit)
    explicit_rvq: Optional[ExplicitRVQ] = None


def look_at(eye, W: int, H: int, fov_x_deg: float = 60.0) -> Camera:
    """SURVEY §8(d) look-at rule: forward = -eye/|eye|, +x right, +y down, +z forward, horizontal fov."""
    eye = np.asarray(eye, dtype=np.float64)
    f = -eye / np.linalg.norm(eye)
    u0 = np.array([0.0, 1.0, 0.0])
    if abs(float(f @ u0)) > 0.99:
        u0 = np.array([1.0, 0.0, 0.0])
    up = u0 - (u0 @ f) * f
    down = -up / np.linalg.norm(up)
    right = np.cross(down, f)
    R = np.stack([right, down, f]).astype(np.float32)
    t = (-(R.astype(np.float64) @ eye)).astype(np.float32)
    fx = W / (2.0 * math.tan(math.radians(fov_x_deg) / 2.0))
    return Camera(R=R, t=t, fx=float(np.float32(fx)), fy=float(np.float32(fx)),
                  cx=(W - 1) / 2.0, cy=(H - 1) / 2.0, W=W, H=H)


def _xavier(rng: np.random.Generator, spec: MlpSpec) -> np.ndarray:
    parts = []
    for o, i in spec.layer_shapes():
        a = math.sqrt(6.0 / (i + o))
        parts.append(rng.uniform(-a, a, size=(o, i)).astype(np.float32).ravel())
    return np.concatenate(parts)


def _table(rng: np.random.Generator, grid: GridSpec, amp: float) -> np.ndarray:
    return rng.uniform(-amp, amp, size=(grid.n_entries(), grid.feats)).astype(np.float32)


def _attrs(rng: np.random.Generator, n: int):
    scale_logit = rng.normal(-4.0, 0.5, size=n).astype(np.float32)
    opacity_logit = rng.normal(0.0, 1.0, size=n).astype(np.float32)
    c = np.clip(rng.uniform(0.0, 1.0, size=(3, n)), 1e-3, 1.0 - 1e-3)
    rgb_logit = np.log(c / (1.0 - c)).astype(np.float32)
    return rgb_logit, scale_logit, opacity_logit


def _unit(v: np.ndarray) -> np.ndarray:
    return v / np.linalg.norm(v, axis=-1, keepdims=True)


def _positions(cfg: int, rng: np.random.Generator, n: int) -> np.ndarray:
    if cfg in (1, 2, 5):
        return rng.uniform(-1.0, 1.0, size=(n, 3))
    if cfg == 3:
        n_far = n // 10
        n_cl = n - n_far
        centres = rng.uniform(-2.0, 2.0, size=(64, 3))
        sig = rng.uniform(0.05, 0.3, size=(64, 3))
        member = rng.integers(0, 64, size=n_cl)
        p_cl = centres[member] + sig[member] * rng.normal(size=(n_cl, 3))
        p_far = 50.0 * _unit(rng.normal(size=(n_far, 3)))
        p = np.concatenate([p_cl, p_far])
        return p[rng.permutation(n)]           # a trained model's order is arbitrary
    if cfg == 4:
        n_far = n // 5
        n_in = n - n_far
        d = _unit(rng.normal(size=(n_in, 3)))
        rad = rng.uniform(0.0, 1.0, size=(n_in, 1)) ** (1.0 / 3.0)
        p_in = d * rad * np.array([2.0, 1.0, 2.0])
        r_far = np.exp(rng.uniform(math.log(2.0), math.log(100.0), size=(n_far, 1)))
        p_far = _unit(rng.normal(size=(n_far, 3))) * r_far
        p = np.concatenate([p_in, p_far])
        return p[rng.permutation(n)]
    raise ValueError(f"unknown config {cfg}")


_DEFAULT_N = {1: 4096, 2: 100_000, 3: 1_000_000, 4: 2_000_000, 5: 500_000}
_DEFAULT_RES = {1: (128, 128), 2: (512, 512), 3: (1280, 720), 4: (1245, 825), 5: (1920, 1080)}


def make_scene(cfg: int, n_gaussians: Optional[int] = None, *, width: Optional[int] = None,
               height: Optional[int] = None, table_amp: float = 0.1, fp16: Optional[bool] = None,
               n_cameras: Optional[int] = None, seed: Optional[int] = None) -> Scene:
    """Build config `cfg` (1..5, BASELINE.json order). `n_gaussians`, `width`, `height`, `n_cameras` scale the
    same recipe down (parity cases) or across config 5's sweep; `table_amp=1.0` gives the "high-gain" scene of
    SURVEY §8(c) H5; `fp16` overrides the config's parameter dtype."""
    if cfg not in _DEFAULT_N:
        raise ValueError(f"unknown config {cfg}")
    n = int(n_gaussians if n_gaussians is not None else _DEFAULT_N[cfg])
    W, H = _DEFAULT_RES[cfg]
    W = int(width if width is not None else W)
    H = int(height if height is not None else H)
    rng = np.random.default_rng(np.random.PCG64(1000 + cfg if seed is None else seed))

    pos = _positions(cfg, rng, n).astype(np.float32)
    rgb_logit, scale_logit, opacity_logit = _attrs(rng, n)

    if cfg == 1:
        geo_grid = GridSpec(list(RES_8), 14)
        app_grid = GridSpec(list(RES_8), 14)
        bg_grid = GridSpec(list(RES_BG4), 14)
        geo_mlp = MlpSpec(geo_grid.levels * 2, 32, 1, 8)
        app_mlp = MlpSpec(app_grid.levels * 2 + PE_DIMS, 32, 1, 3)
        bg_mlp = MlpSpec(bg_grid.levels * 2 + PE_DIMS, 32, 1, 3)
    else:
        geo_grid = GridSpec(list(RES_16), 19)
        app_grid = GridSpec(list(RES_16), 19)
        bg_grid = GridSpec(list(RES_BG8), 19)
        geo_mlp = MlpSpec(geo_grid.levels * 2, 64, 2, 8)
        app_mlp = MlpSpec(app_grid.levels * 2 + PE_DIMS, 64, 2, 3)
        bg_mlp = MlpSpec(bg_grid.levels * 2 + PE_DIMS, 64, 1, 3)

    geo_table = _table(rng, geo_grid, table_amp)
    app_table = _table(rng, app_grid, table_amp)
    bg_table = _table(rng, bg_grid, table_amp)
    geo_w = _xavier(rng, geo_mlp)
    app_w = _xavier(rng, app_mlp)
    bg_w = _xavier(rng, bg_mlp)

    use_fp16 = (cfg >= 3) if fp16 is None else bool(fp16)
    if use_fp16:
        geo_table, app_table, bg_table = (a.astype(np.float16) for a in (geo_table, app_table, bg_table))
        geo_w, app_w, bg_w = (a.astype(np.float16) for a in (geo_w, app_w, bg_w))

    half = 1.0 if cfg in (1, 2, 5) else 2.0
    scene = Scene(
        name=f"cfg{cfg}_n{n}_{W}x{H}_{'f16' if use_fp16 else 'f32'}", n=n,
        pos=np.ascontiguousarray(pos.T), rgb_logit=np.ascontiguousarray(rgb_logit),
        scale_logit=scale_logit, opacity_logit=opacity_logit,
        aabb_min=np.full(3, -half, np.float32), aabb_max=np.full(3, half, np.float32),
        geo_grid=geo_grid, app_grid=app_grid, bg_grid=bg_grid,
        geo_mlp=geo_mlp, app_mlp=app_mlp, bg_mlp=bg_mlp,
        geo_table=geo_table, app_table=app_table, bg_table=bg_table,
        geo_w=geo_w, app_w=app_w, bg_w=bg_w, fp16=use_fp16)

    crng = np.random.default_rng(np.random.PCG64((1000 + cfg if seed is None else seed) + 7919))
    if cfg == 1:
        eyes = [np.array([0.0, 0.0, -3.0])]
    elif cfg == 2:
        eyes = list(3.0 * _unit(crng.normal(size=(5, 3))))
    elif cfg == 3:
        eyes = [4.0 * np.array([math.cos(2 * math.pi * k / 20), 0.0, math.sin(2 * math.pi * k / 20)]) for k in range(20)]
    elif cfg == 4:
        eyes = [3.5 * np.array([math.cos(2 * math.pi * k / 60), 0.0, math.sin(2 * math.pi * k / 60)]) for k in range(60)]
    else:
        eyes = [np.array([0.0, 0.0, -3.0])]
    if n_cameras is not None:
        eyes = eyes[:n_cameras]
    scene.cameras = [look_at(e, W, H) for e in eyes]
    return scene


def quantize8(scene: Scene) -> Scene:
    """The post-processing step of PAPER.md:229 (3) applied to a generated scene: every level of every table becomes
    8-bit min-max codes, code = rint((v - min) / step), step = (max - min) / 255, per level and feature. This is the
    ENCODER (input preparation); the decode the renderer performs is defined in DESIGN.md §2 D3'. Weights become fp16."""
    import copy
    s = copy.copy(scene)
    for name, grid in (("geo", scene.geo_grid), ("app", scene.app_grid), ("bg", scene.bg_grid)):
        tab = np.asarray(getattr(scene, name + "_table"), dtype=np.float32)
        codes = np.zeros(tab.shape, np.uint8)
        q = np.zeros((grid.levels, 2, 2), np.float32)
        off = 0
        for l, sz in enumerate(grid.level_sizes()):
            seg = tab[off:off + sz]
            for f in range(2):
                mn, mx = np.float32(seg[:, f].min()), np.float32(seg[:, f].max())
                step = np.float32((mx - mn) / np.float32(255.0)) if mx > mn else np.float32(1.0)
                codes[off:off + sz, f] = np.clip(np.rint((seg[:, f] - mn) / step), 0, 255).astype(np.uint8)
                q[l, f] = (mn, step)
            off += sz
        setattr(s, name + "_table", codes)
        setattr(s, name + "_q", q)
        setattr(s, name + "_w", np.asarray(getattr(scene, name + "_w")).astype(np.float16))
    s.quant8 = True
    s.fp16 = True
    s.name = scene.name + "_q8"
    return s


def compress_explicit(scene: Scene, stages: int = 6, codebook_size: int = 64, seed: int = 0,
                      lloyd_iters: int = 2) -> Scene:
    """The post-processing steps of PAPER.md:229 (1)-(2) applied to a generated scene: positions rounded to binary16,
    the rows (s_e, alpha_e, c_e) residual-vector-quantised: stage s clusters what stages 0..s-1 left over (codebook
    seeded from random rows, a few Lloyd iterations) and stores the nearest row's index. This is the ENCODER (input
    preparation, as quantize8 is); the decode the renderer performs is defined in DESIGN.md §2 D1'."""
    import copy
    rng = np.random.default_rng(np.random.PCG64(90_000 + seed))
    n = scene.n
    rows = np.concatenate([np.asarray(scene.scale_logit, np.float32)[:, None],
                           np.asarray(scene.opacity_logit, np.float32)[:, None],
                           np.asarray(scene.rgb_logit, np.float32).T], axis=1)          # (N, 5)
    K = int(codebook_size)
    books = np.zeros((stages, K, 5), np.float32)
    codes = np.zeros((stages, n), np.uint16)
    resid = rows.copy()

    def nearest(x: np.ndarray, book: np.ndarray) -> np.ndarray:
        out = np.zeros(len(x), np.int64)
        b2 = (book.astype(np.float64) ** 2).sum(1)
        step = max(1, (1 << 22) // len(book))
        for a in range(0, len(x), step):
            blk = x[a:a + step].astype(np.float64)
            out[a:a + step] = np.argmin(b2[None, :] - 2.0 * blk @ book.astype(np.float64).T, axis=1)
        return out

    for st in range(stages):
        book = resid[rng.integers(0, n, size=K)].copy()
        for _ in range(lloyd_iters):
            k = nearest(resid, book)
            cnt = np.bincount(k, minlength=K)
            for d in range(5):
                sums = np.bincount(k, weights=resid[:, d].astype(np.float64), minlength=K)
                book[:, d] = np.where(cnt > 0, sums / np.maximum(cnt, 1), book[:, d]).astype(np.float32)
        k = nearest(resid, book)
        books[st], codes[st] = book, k.astype(np.uint16)
        resid = (resid - book[k]).astype(np.float32)
    s = copy.copy(scene)
    s.explicit_rvq = ExplicitRVQ(pos_h=np.ascontiguousarray(np.asarray(scene.pos, np.float32).astype(np.float16).view(np.uint16)),
                                 codes=codes, codebooks=books)
    s.name = scene.name + f"_rvq{stages}x{K}"
    return s


def tiny_scene(n: int = 48, W: int = 32, H: int = 32, seed: int = 7, fp16: bool = False, levels: int = 4,
               log2_table: int = 10, hidden: int = 16, n_hidden: int = 1, table_amp: float = 0.5,
               scale_mean: float = -2.5) -> Scene:
    """A very small scene for brute-force pins (<=64 Gaussians, <=32x32 px). Bigger splats and a
    hash table small enough that both dense and hashed levels occur."""
    rng = np.random.default_rng(np.random.PCG64(seed))
    pos = rng.uniform(-1.0, 1.0, size=(n, 3)).astype(np.float32)
    rgb_logit, _, opacity_logit = _attrs(rng, n)
    scale_logit = rng.normal(scale_mean, 0.5, size=n).astype(np.float32)
    res = [4, 7, 12, 21, 37, 64, 111, 192][:levels]
    grid = GridSpec(res, log2_table)
    bg_grid = GridSpec(res[: max(2, levels // 2)], log2_table)
    geo_mlp = MlpSpec(grid.levels * 2, hidden, n_hidden, 8)
    app_mlp = MlpSpec(grid.levels * 2 + PE_DIMS, hidden, n_hidden, 3)
    bg_mlp = MlpSpec(bg_grid.levels * 2 + PE_DIMS, hidden, 1, 3)
    tabs = [_table(rng, g, table_amp) for g in (grid, grid, bg_grid)]
    ws = [_xavier(rng, m) for m in (geo_mlp, app_mlp, bg_mlp)]
    if fp16:
        tabs = [a.astype(np.float16) for a in tabs]
        ws = [a.astype(np.float16) for a in ws]
    s = Scene(name=f"tiny_n{n}_{W}x{H}", n=n, pos=np.ascontiguousarray(pos.T), rgb_logit=rgb_logit,
              scale_logit=scale_logit, opacity_logit=opacity_logit,
              aabb_min=np.full(3, -1.0, np.float32), aabb_max=np.full(3, 1.0, np.float32),
              geo_grid=grid, app_grid=GridSpec(list(res), log2_table), bg_grid=bg_grid,
              geo_mlp=geo_mlp, app_mlp=app_mlp, bg_mlp=bg_mlp,
              geo_table=tabs[0], app_table=tabs[1], bg_table=tabs[2],
              geo_w=ws[0], app_w=ws[1], bg_w=ws[2], fp16=fp16)
    s.cameras = [look_at(np.array([0.0, 0.0, -3.0]), W, H), look_at(np.array([2.0, 1.0, 2.0]), W, H)]
    return s


def morton_sorted(scene: Scene) -> Scene:
    """The same scene with its Gaussians stored in Morton (Z-curve) order of their positions: SURVEY §8(d)'s secondary,
    labelled measurement (a trained model's order is arbitrary, so the order as generated stays the primary one). A pure
    permutation of the input arrays: 10 bits per axis over the bounding box of the positions."""
    import copy
    pos = np.asarray(scene.pos, np.float32)
    lo, hi = pos.min(axis=1, keepdims=True), pos.max(axis=1, keepdims=True)
    q = np.clip(((pos - lo) / np.maximum(hi - lo, 1e-30) * 1023.0).astype(np.uint64), 0, 1023)

    def spread(v):
        v = (v | (v << np.uint64(16))) & np.uint64(0x030000FF)
        v = (v | (v << np.uint64(8))) & np.uint64(0x0300F00F)
        v = (v | (v << np.uint64(4))) & np.uint64(0x030C30C3)
        v = (v | (v << np.uint64(2))) & np.uint64(0x09249249)
        return v

    code = spread(q[0]) | (spread(q[1]) << np.uint64(1)) | (spread(q[2]) << np.uint64(2))
    order = np.argsort(code, kind="stable")
    s = copy.copy(scene)
    s.pos = np.ascontiguousarray(pos[:, order])
    s.rgb_logit = np.ascontiguousarray(np.asarray(scene.rgb_logit)[:, order])
    s.scale_logit = np.ascontiguousarray(np.asarray(scene.scale_logit)[order])
    s.opacity_logit = np.ascontiguousarray(np.asarray(scene.opacity_logit)[order])
    s.name = scene.name + "_morton"
    return s


def shard_cameras(n_cameras: int, rank: int, world: int) -> List[int]:
    """Frame-parallel replicas: cameras dealt round-robin, no collective on the data path."""
    return list(range(rank, n_cameras, world))


def strip_rows(H: int, rank: int, world: int, align: int = 64):
    """Screen-strip parallelism: pixel rows [begin, end) of rank `rank` of `world`. Strips are equal
    multiples of `align` rows (64 = one macro tile of 4 x 4 tiles, so that no macro-tile list is binned twice), the
    last one takes what is left; a rank beyond the image gets an empty strip (begin == end == H)."""
    units = (H + align - 1) // align
    per = (units + world - 1) // world
    begin = min(rank * per * align, H)
    end = min((rank + 1) * per * align, H)
    return begin, end
