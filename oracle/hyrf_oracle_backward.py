"""CPU oracle of the BACKWARD pass (§3.4, Eq. 12): float64, plain PyTorch CPU ops.

TEST INFRASTRUCTURE, NOT PRODUCT (same rules as hyrf_oracle.py: only tests/, smoke() and bench.py's CPU legs import it;
it never imports the CUDA binding and shares no code with csrc/).

What is differentiated. The forward pass is discontinuous (cull, cell indices, 3-sigma rectangles, alpha < 1/255 skip,
T' < 1e-4 stop, min(0.99, .) clamp, tau_T test, ReLU, contraction branch): as in the training of the rasterizer the
paper builds on, every such DECISION is frozen at what the binary32 forward pass
(hyrf_oracle.c) took, and the smooth arithmetic in between is differentiated exactly:

    loss (Eq. 12)  <-  out = C_fg + T c_s (Eq. 10-11)  <-  alpha blend (Eq. 1; hyrf_oracle.c ho_stage_raster_backward)
                   <-  EWA projection (D8)  <-  aggregation (Eq. 7)  <-  decoders (Eq. 4, 6)  <-  grid encodes (Eq. 3),
                       direction encoding (Eq. 5), contraction (Eq. 2)  <-  explicit Gaussians, tables, weights.

How. Stages S2-S4a and S6 are RESTATED here in float64 torch ops, formula by formula from DESIGN.md §2 (D2-D8, D11), and
their vector-Jacobian products come from torch.autograd: the gradient of a restated formula is its definition. The
restatement is pinned against the C oracle's forward values (tests/test_oracle_backward.py), so a slip in it shows up
as a forward mismatch; the chain as a whole is pinned by central differences of the C oracle's full render. Roundings to
binary16 (fp16 configs: features, hidden activations) are identities for the gradient (straight-through), the float64
forward simply omits them.

Reading A28: L = (1 - lambda) L1 + lambda (1 - SSIM), lambda = 0.2, SSIM with an 11 x 11 Gaussian window
(sigma 1.5), C1 = 0.01^2, C2 = 0.03^2, zero padding, mean over pixels and channels — "the same L1 loss and SSIM loss as
the original 3DGS".
"""
from __future__ import annotations

import math
from typing import Dict, Optional

import numpy as np
import torch

from . import hyrf_oracle as ho

F64 = torch.float64
PRIME_Y, PRIME_Z = 2654435761, 805459861


def _t(a, grad: bool = False) -> torch.Tensor:
    t = torch.from_numpy(np.ascontiguousarray(np.asarray(a, dtype=np.float64)))
    return t.requires_grad_(True) if grad else t


class Params:
    """The trainable parameters of a scene as float64 leaf tensors: explicit Gaussians, the three grid
    tables, the three decoders. 8-bit tables are differentiated through their decoded values."""

    def __init__(self, scene):
        if getattr(scene, "explicit_rvq", None) is not None:
            scene = ho.with_decoded_explicit(scene)
        self.scene = scene
        self.pos = _t(scene.pos, True)                       # (3, N)
        self.scale_logit = _t(scene.scale_logit, True)       # (N,)
        self.opacity_logit = _t(scene.opacity_logit, True)   # (N,)
        self.rgb_logit = _t(scene.rgb_logit, True)           # (3, N)
        if getattr(scene, "quant8", False):
            raise ValueError("the backward oracle takes plain (fp32 / fp16) tables")
        self.geo_table = _t(np.asarray(scene.geo_table, np.float32), True)
        self.app_table = _t(np.asarray(scene.app_table, np.float32), True)
        self.bg_table = _t(np.asarray(scene.bg_table, np.float32), True)
        self.geo_w = _t(np.asarray(scene.geo_w, np.float32), True)
        self.app_w = _t(np.asarray(scene.app_w, np.float32), True)
        self.bg_w = _t(np.asarray(scene.bg_w, np.float32), True)

    def leaves(self) -> Dict[str, torch.Tensor]:
        return dict(pos=self.pos, scale_logit=self.scale_logit, opacity_logit=self.opacity_logit, rgb_logit=self.rgb_logit,
                    geo_table=self.geo_table, app_table=self.app_table, bg_table=self.bg_table,
                    geo_w=self.geo_w, app_w=self.app_w, bg_w=self.bg_w)


# ---------------------------------------------------------------------------------------------- D2 contraction
def contract(p: torch.Tensor, amin, amax) -> torch.Tensor:
    """p (V, 3) world positions -> x (V, 3) in [0, 1]^3 (Eq. 2 / 13-14 with reading A1)."""
    c = 0.5 * (_t(amin) + _t(amax))
    h = 0.5 * (_t(amax) - _t(amin))
    q = (p - c) / h
    n = torch.sqrt((q * q).sum(-1, keepdim=True))
    outside = n > 1.0
    n_safe = torch.where(outside, n, torch.ones_like(n))
    q = torch.where(outside, (2.0 - 1.0 / n_safe) / n_safe * q, q)
    return torch.clamp(0.25 * q + 0.5, 0.0, 1.0)


# ---------------------------------------------------------------------------------------------- D3 grid encode
def cells_fp32(grid, x32: np.ndarray):
    """The cells the binary32 forward pass picks (D3: u = x N in binary32, i = min(floor(u), N - 1)), per level (V, 3)."""
    out = []
    for N in grid.level_res:
        u = (x32.astype(np.float32) * np.float32(N)).astype(np.float32)
        out.append(torch.from_numpy(np.minimum(np.floor(u), N - 1).astype(np.int64)))
    return out


def grid_encode(grid, table: torch.Tensor, x: torch.Tensor, cells=None) -> torch.Tensor:
    """x (V, 3) -> features (V, 2 L), level-major [l][f] (Eq. 3; layout and hash of DESIGN.md §2 D3). The cell
    (integer part) is a frozen decision — `cells` (from cells_fp32) when given, else taken from x itself; the weights
    are differentiable in x, the values in the table."""
    _, sizes, offs, dense = ho.grid_layout(grid)
    T = 1 << grid.log2_table
    feats = []
    for l, N in enumerate(grid.level_res):
        u = x * float(N)
        i = cells[l] if cells is not None else torch.clamp(torch.floor(u.detach()), max=float(N - 1)).to(torch.int64)       # (V, 3)
        w = u - i.to(F64)
        acc = torch.zeros((x.shape[0], 2), dtype=F64)
        for k in range(8):
            b = [(k >> a) & 1 for a in range(3)]
            v = [i[:, a] + b[a] for a in range(3)]
            if dense[l]:
                idx = v[0] + (N + 1) * (v[1] + (N + 1) * v[2])
            else:
                idx = ((v[0] ^ ((v[1] * PRIME_Y) & 0xFFFFFFFF) ^ ((v[2] * PRIME_Z) & 0xFFFFFFFF)) & 0xFFFFFFFF) & (T - 1)
            wt = ((w[:, 0] if b[0] else 1.0 - w[:, 0]) * (w[:, 1] if b[1] else 1.0 - w[:, 1])) * (w[:, 2] if b[2] else 1.0 - w[:, 2])
            acc = acc + wt[:, None] * table[int(offs[l]) + idx]
        feats.append(acc)
    return torch.cat(feats, dim=1)


# ---------------------------------------------------------------------------------------------- D4 direction encoding
def dir_pe(d: torch.Tensor, octaves: int) -> torch.Tensor:
    """d (V, 3) unit vectors -> (V, 6 K): index 6k + a = sin(pi 2^k d_a), 6k + 3 + a = cos(...) (Eq. 5, reading A10)."""
    out = []
    for k in range(octaves):
        ang = math.pi * float(1 << k) * d
        out += [torch.sin(ang), torch.cos(ang)]
    return torch.cat(out, dim=1)


# ---------------------------------------------------------------------------------------------- D5 MLP
def relu_masks_fp32(spec, w32: np.ndarray, x32: np.ndarray, fp16: bool):
    """Which hidden units the binary32 forward pass (hyrf_oracle.c ho_mlp_forward, D5's fma order) leaves on: one (V, hidden)
    0 / 1 array per hidden layer. Hidden layer l is read out through a decoder truncated after it whose output layer
    is the identity (fma with 1 and 0 is exact)."""
    import types
    V = x32.shape[0]
    dims = [spec.in_dim] + [spec.hidden] * spec.n_hidden
    masks, off = [], 0
    eye = np.eye(spec.hidden, dtype=np.float32).ravel()
    for l in range(spec.n_hidden):
        off += dims[l + 1] * dims[l]
        sub = types.SimpleNamespace(in_dim=spec.in_dim, hidden=spec.hidden, n_hidden=l + 1, out_dim=spec.hidden)
        wl = np.concatenate([np.asarray(w32[:off], np.float32), eye])
        h = np.stack([ho.mlp_forward(sub, wl, x32[v], fp16) for v in range(V)]) if V else np.zeros((0, spec.hidden), np.float32)
        masks.append(torch.from_numpy((h > 0).astype(np.float64)))
    return masks


def mlp(spec, w: torch.Tensor, x: torch.Tensor, masks=None) -> torch.Tensor:
    """in -> hidden x n_hidden (ReLU) -> out (linear), no biases; weights flat, layers concatenated, row-major [out][in]
    (Eq. 4, 6; reading A11). x is zero-padded to in_dim. `masks` (from relu_masks_fp32): the ReLU decisions
    of the binary32 forward pass, frozen; else the float64 values decide."""
    if x.shape[1] < spec.in_dim:
        x = torch.cat([x, torch.zeros((x.shape[0], spec.in_dim - x.shape[1]), dtype=F64)], dim=1)
    dims = [spec.in_dim] + [spec.hidden] * spec.n_hidden + [spec.out_dim]
    off = 0
    h = x
    for li in range(len(dims) - 1):
        o, i = dims[li + 1], dims[li]
        W = w[off:off + o * i].reshape(o, i)
        off += o * i
        h = h @ W.T
        if li < len(dims) - 2:
            h = h * masks[li] if masks is not None else torch.relu(h)
    return h


# ---------------------------------------------------------------------------------------------- D7 aggregation
def aggregate(raw: torch.Tensor, s_e, a_e, c_e) -> torch.Tensor:
    """raw (V, 11) = (alpha_n, s_n[3], r_n[4], c_n[3]) + explicit (s_e (V,), alpha_e (V,), c_e (V, 3)) -> attrs (V, 11) =
    (s[3], r[4] wxyz, alpha, c[3]) (Eq. 7)."""
    s = torch.sigmoid(raw[:, 1:4] + s_e[:, None])
    m = torch.sqrt((raw[:, 4:8] ** 2).sum(-1, keepdim=True))
    r = raw[:, 4:8] / torch.clamp(m, min=1e-12)
    alpha = torch.sigmoid(raw[:, 0:1] + a_e[:, None])
    c = torch.sigmoid(raw[:, 8:11] + c_e)
    return torch.cat([s, r, alpha, c], dim=1)


# ---------------------------------------------------------------------------------------------- D8 projection
def project(attrs: torch.Tensor, p: torch.Tensor, cam) -> torch.Tensor:
    """attrs (V, 11), world positions p (V, 3) -> differentiable part of the projected record (V, 9) =
    (u, v, A, B, C, opacity, r, g, b) (EWA, DESIGN.md §2 D8). Depth, radius and the tile rectangle carry no gradient."""
    R = _t(np.asarray(cam.R, np.float32).reshape(3, 3))
    t = _t(np.asarray(cam.t, np.float32).reshape(3))
    fx, fy, cx, cy = float(np.float32(cam.fx)), float(np.float32(cam.fy)), float(np.float32(cam.cx)), float(np.float32(cam.cy))
    s, q = attrs[:, 0:3], attrs[:, 3:7]
    w, x, y, z = q[:, 0], q[:, 1], q[:, 2], q[:, 3]
    M = torch.stack([
        torch.stack([1 - 2 * (y * y + z * z), 2 * (x * y - w * z), 2 * (x * z + w * y)], -1),
        torch.stack([2 * (x * y + w * z), 1 - 2 * (x * x + z * z), 2 * (y * z - w * x)], -1),
        torch.stack([2 * (x * z - w * y), 2 * (y * z + w * x), 1 - 2 * (x * x + y * y)], -1)], 1)   # (V, 3, 3)
    L = M * s[:, None, :]
    Sigma = L @ L.transpose(1, 2)
    pc = p @ R.T + t
    X, Y, Z = pc[:, 0], pc[:, 1], pc[:, 2]
    iz = 1.0 / Z
    xn, yn = X * iz, Y * iz
    zero = torch.zeros_like(iz)
    J = torch.stack([torch.stack([fx * iz, zero, -(fx * xn) * iz], -1),
                     torch.stack([zero, fy * iz, -(fy * yn) * iz], -1)], 1)                          # (V, 2, 3)
    Tm = J @ R
    cov = Tm @ Sigma @ Tm.transpose(1, 2)
    a, b, c = cov[:, 0, 0] + 0.3, cov[:, 0, 1], cov[:, 1, 1] + 0.3
    det = a * c - b * b
    A, B, C = c / det, -b / det, a / det
    u, v = fx * xn + cx, fy * yn + cy
    return torch.stack([u, v, A, B, C, attrs[:, 7], attrs[:, 8], attrs[:, 9], attrs[:, 10]], -1)


def fields_forward(P: Params, cam, vis_idx: np.ndarray, ablation: int = 0, frozen: bool = False):
    """Stages S2-S4a for the visible Gaussians in float64: returns (raw (V, 11), attrs (V, 11), rec (V, 9)). frozen: the
    grid cells and ReLU masks are those of the binary32 forward pass (what the backward pass differentiates around);
    otherwise the float64 values decide (the two differ for a Gaussian in a few thousand)."""
    sc = P.scene
    idx = torch.from_numpy(np.asarray(vis_idx, np.int64))
    p = P.pos[:, idx].T                                              # (V, 3)
    x = contract(p, sc.aabb_min, sc.aabb_max)
    if ablation & ho.ABL_NO_NEURAL:
        raw = torch.zeros((len(idx), 11), dtype=F64)
    else:
        cg = ca = mg = ma = None
        if frozen:
            # the decisions of the binary32 forward pass: cells of every level, ReLU masks of both decoders
            fp16 = bool(sc.fp16)
            pos32 = np.asarray(sc.pos, np.float32)[:, np.asarray(vis_idx, np.int64)].T
            x32 = np.stack([ho.contract(q, sc.aabb_min, sc.aabb_max) for q in pos32]) if len(pos32) else np.zeros((0, 3), np.float32)
            cg, ca = cells_fp32(sc.geo_grid, x32), cells_fp32(sc.app_grid, x32)
            o32 = ho.camera_center(cam)
            fg = np.stack([ho.grid_encode(sc.geo_grid, sc.geo_table, q, fp16) for q in x32])
            fa = np.stack([np.concatenate([ho.grid_encode(sc.app_grid, sc.app_table, q, fp16),
                                           ho.dir_pe(ho.view_dir(pp, o32), sc.dir_pe_octaves, fp16)]) for q, pp in zip(x32, pos32)])
            pad = lambda a, n: np.concatenate([a, np.zeros((a.shape[0], n - a.shape[1]), np.float32)], 1) if a.shape[1] < n else a
            mg = relu_masks_fp32(sc.geo_mlp, np.asarray(sc.geo_w, np.float32), pad(fg, sc.geo_mlp.in_dim), fp16)
            ma = relu_masks_fp32(sc.app_mlp, np.asarray(sc.app_w, np.float32), pad(fa, sc.app_mlp.in_dim), fp16)
        f_geo = grid_encode(sc.geo_grid, P.geo_table, x, cg)
        f_app = grid_encode(sc.app_grid, P.app_table, x, ca)
        o = _t(ho.camera_center(cam))
        delta = p - o
        d = delta / torch.sqrt((delta * delta).sum(-1, keepdim=True))
        raw = torch.cat([mlp(sc.geo_mlp, P.geo_w, f_geo, mg),
                         mlp(sc.app_mlp, P.app_w, torch.cat([f_app, dir_pe(d, sc.dir_pe_octaves)], dim=1), ma)], dim=1)
    if ablation & ho.ABL_NO_EXPLICIT:
        z = torch.zeros(len(idx), dtype=F64)
        attrs = aggregate(raw, z, z, torch.zeros((len(idx), 3), dtype=F64))
    else:
        attrs = aggregate(raw, P.scale_logit[idx], P.opacity_logit[idx], P.rgb_logit[:, idx].T)
    return raw, attrs, project(attrs, p, cam)


# ---------------------------------------------------------------------------------------------- D11 background
def background_colors(P: Params, cam, pix: np.ndarray, frozen: bool = False) -> torch.Tensor:
    """c_s (n, 3) for the pixels pix (n, 2) = (i, j) (PAPER.md:124-134 Eq. 10-11, :360-378 Eq. 15-18; D11)."""
    sc = P.scene
    R = _t(np.asarray(cam.R, np.float32).reshape(3, 3))
    o = _t(ho.camera_center(cam))
    ij = _t(pix)
    dc = torch.stack([(ij[:, 0] - float(np.float32(cam.cx))) / float(np.float32(cam.fx)),
                      (ij[:, 1] - float(np.float32(cam.cy))) / float(np.float32(cam.fy)), torch.ones(len(ij), dtype=F64)], -1)
    dw = dc @ R                                                      # R^T dc
    d = dw / torch.sqrt((dw * dw).sum(-1, keepdim=True))
    Bq = 2.0 * (d @ o)
    Cq = (o * o).sum() - float(np.float32(sc.bg_radius)) ** 2
    tt = 0.5 * (-Bq + torch.sqrt(Bq * Bq - 4.0 * Cq))
    ps = o + tt[:, None] * d
    x = contract(ps, sc.aabb_min, sc.aabb_max)
    cells = masks = None
    if frozen and len(pix):
        fp16 = bool(sc.fp16)
        rays = [ho.ray_sphere(cam, float(i), float(j), float(sc.bg_radius)) for i, j in pix]
        x32 = np.stack([ho.contract(ps32, sc.aabb_min, sc.aabb_max) for _, ps32 in rays])
        cells = cells_fp32(sc.bg_grid, x32)
        fin = np.stack([np.concatenate([ho.grid_encode(sc.bg_grid, sc.bg_table, q, fp16), ho.dir_pe(d32, sc.dir_pe_octaves, fp16)])
                        for q, (d32, _) in zip(x32, rays)])
        if fin.shape[1] < sc.bg_mlp.in_dim:
            fin = np.concatenate([fin, np.zeros((fin.shape[0], sc.bg_mlp.in_dim - fin.shape[1]), np.float32)], 1)
        masks = relu_masks_fp32(sc.bg_mlp, np.asarray(sc.bg_w, np.float32), fin, fp16)
    f = grid_encode(sc.bg_grid, P.bg_table, x, cells)
    return torch.sigmoid(mlp(sc.bg_mlp, P.bg_w, torch.cat([f, dir_pe(d, sc.dir_pe_octaves)], dim=1), masks))


# ---------------------------------------------------------------------------------------------- Eq. 12 loss
def _ssim_window() -> torch.Tensor:
    g = torch.tensor([math.exp(-((k - 5) ** 2) / (2.0 * 1.5 ** 2)) for k in range(11)], dtype=F64)
    g = g / g.sum()
    return (g[:, None] * g[None, :])[None, None]


def ssim(a: torch.Tensor, b: torch.Tensor) -> torch.Tensor:
    """Mean SSIM of two (H, W, 3) images: 11 x 11 Gaussian window (sigma 1.5), C1 = 0.01^2, C2 = 0.03^2, zero padding."""
    win = _ssim_window().expand(3, 1, 11, 11)
    A, Bm = a.permute(2, 0, 1)[None], b.permute(2, 0, 1)[None]
    conv = lambda t: torch.nn.functional.conv2d(t, win, padding=5, groups=3)
    mu_a, mu_b = conv(A), conv(Bm)
    s_aa, s_bb, s_ab = conv(A * A) - mu_a * mu_a, conv(Bm * Bm) - mu_b * mu_b, conv(A * Bm) - mu_a * mu_b
    C1, C2 = 0.01 ** 2, 0.03 ** 2
    m = ((2 * mu_a * mu_b + C1) * (2 * s_ab + C2)) / ((mu_a * mu_a + mu_b * mu_b + C1) * (s_aa + s_bb + C2))
    return m.mean()


def loss_l1_ssim(img: torch.Tensor, gt: torch.Tensor, lam: float = 0.2) -> torch.Tensor:
    """PAPER.md:138-140 Eq. 12 (reading A28)."""
    return (1.0 - lam) * (img - gt).abs().mean() + lam * (1.0 - ssim(img, gt))


def loss_and_grad(img: np.ndarray, gt: np.ndarray, lam: float = 0.2):
    """(L, dL/d img) for (H, W, 3) images."""
    x = _t(img, True)
    L = loss_l1_ssim(x, _t(gt), lam)
    L.backward()
    return float(L.detach()), x.grad.numpy().copy()


# ---------------------------------------------------------------------------------------------- the whole chain
def backward_from_image_grad(scene, cam, g_out: np.ndarray, ablation: int = 0, fwd: Optional[dict] = None):
    """Gradients of a scalar L with respect to every parameter, given g_out = dL/d out (H, W, 3), for one camera.

    Decisions come from the binary32 forward pass (`fwd` = hyrf_oracle.render(...), computed here when not given): visible
    set, per-tile lists, the blended prefix of every pixel, the background mask. Steps, back to front:
      S6  out = C_fg + T c_s on the mask  ->  g_Cfg = g_out,  g_T = sum_c g_out c_s,  g_cs = T g_out  -> bg table / weights
      S5  hyrf_oracle.c ho_stage_raster_backward (float64 on the frozen blended sets)  ->  g_rec (V, 9)
      S4a-S2  autograd of the float64 restatement above  ->  explicit parameters, geo / app tables and weights.
    Returns dict(name -> float64 numpy array shaped like the parameter), plus "g_rec", "g_T" for stage-level tests."""
    osc = ho.OracleScene(scene)
    W, H = int(cam.W), int(cam.H)
    if fwd is None:
        fwd = ho.render(osc, cam, ablation=ablation)
    P = Params(scene)
    g_out_t = _t(g_out).reshape(H, W, 3)
    # ---- S6
    mask = fwd["bg_mask"].astype(bool)
    g_T = np.zeros((H, W), np.float64)
    scalar = torch.zeros((), dtype=F64)
    if mask.any():
        jj, ii = np.nonzero(mask)
        cs = background_colors(P, cam, np.stack([ii, jj], -1).astype(np.float64), frozen=True)
        Tm = _t(fwd["T"][mask])
        g_sel = g_out_t[torch.from_numpy(jj), torch.from_numpy(ii)]
        g_T[mask] = (g_sel * cs.detach()).sum(-1).numpy()
        scalar = scalar + (g_sel * Tm[:, None] * cs).sum()
    # ---- S5 (frozen decisions, float64)
    V = len(fwd["vis_idx"])
    g_rec = ho.stage_raster_backward(W, H, fwd["proj"], fwd["list_rank"], fwd["ranges"],
                                     np.asarray(g_out, np.float32).reshape(H, W, 3), g_T.astype(np.float32)) if V else np.zeros((0, 9))
    # ---- S4a .. S2
    if V:
        _, _, rec = fields_forward(P, cam, fwd["vis_idx"], ablation, frozen=True)
        live = torch.from_numpy((fwd["tiles"] > 0).astype(np.float64))[:, None]      # dropped Gaussians are in no list
        scalar = scalar + (rec * _t(g_rec) * live).sum()
    grads = {k: np.zeros(tuple(v.shape)) for k, v in P.leaves().items()}
    if scalar.requires_grad:
        scalar.backward()
        for k, v in P.leaves().items():
            if v.grad is not None:
                grads[k] = v.grad.numpy().copy()
    grads["g_rec"] = g_rec
    grads["g_T"] = g_T
    return grads


def training_backward(scene, cam, gt: np.ndarray, lam: float = 0.2, ablation: int = 0):
    """One training step's loss and gradients for one camera: L of Eq. 12 between the binary32 render
    and `gt`, then backward_from_image_grad. Returns (L, grads)."""
    fwd = ho.render(ho.OracleScene(scene), cam, ablation=ablation)
    L, g_out = loss_and_grad(fwd["out"], gt, lam)
    return L, backward_from_image_grad(scene, cam, g_out, ablation, fwd)
