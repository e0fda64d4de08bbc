"""Pins for D12, the backward of the alpha blend (oracle ho_stage_raster_backward; DESIGN.md §2 D12). Expected values
come from hand-worked single-pair cases, from torch autograd (float64) on a blend written with torch ops, and from
central finite differences of the oracle's FORWARD stage — never from the backward itself."""
import numpy as np
import pytest


def _one(u, v, A, B, C, o, rgb, depth=1.0):
    return np.array([[u, v, depth, A, B, C, o, *rgb]], np.float32)


def _lists(W, H, n):
    gx, gy = (W + 15) // 16, (H + 15) // 16
    ranges = np.zeros((gx * gy, 2), np.uint32)
    ranges[:, 0] = np.arange(gx * gy) * n
    ranges[:, 1] = ranges[:, 0] + n
    return np.tile(np.arange(n, dtype=np.uint32), gx * gy), ranges


def test_single_pair_at_the_centre_hand_values(ho):
    # one Gaussian centred on pixel (3, 2) of a 16 x 16 image, gradient only at that pixel: dx = dy = 0, alpha = o,
    # C = c o, T = 1 - o  =>  dL/dc = o gC, dL/do = gC . c - gT; position and conic get nothing (power is stationary)
    proj = _one(3.0, 2.0, 0.5, 0.1, 0.4, 0.25, (0.2, 0.6, 0.9))
    lr, rg = _lists(16, 16, 1)
    gc = np.zeros((16, 16, 3), np.float32)
    gt = np.zeros((16, 16), np.float32)
    gc[2, 3] = (1.0, 2.0, -1.0)
    gt[2, 3] = 0.25
    g = ho.stage_raster_backward(16, 16, proj, lr, rg, gc, gt)[0]
    assert np.allclose(g[6:9], 0.25 * np.array([1.0, 2.0, -1.0]), rtol=1e-6)
    assert np.isclose(g[5], 0.2 * 1 + 0.6 * 2 - 0.9 * 1 - 0.25, rtol=1e-6)
    assert np.abs(g[:5]).max() < 1e-12


def test_single_pair_off_centre_hand_values(ho):
    # pixel (5, 2), mean (3, 2): dx = -2, dy = 0, power = -0.5 A 4 = -2 A; with A = 0.25: G = exp(-0.5), alpha = o G
    A, o, c = 0.25, 0.5, 0.8
    proj = _one(3.0, 2.0, A, 0.3, 0.7, o, (c, 0.0, 0.0))
    lr, rg = _lists(16, 16, 1)
    gc = np.zeros((16, 16, 3), np.float32)
    gc[2, 5, 0] = 1.0
    g = ho.stage_raster_backward(16, 16, proj, lr, rg, gc, np.zeros((16, 16), np.float32))[0]
    G = np.exp(-0.5)
    dP = c * o * G                                   # dL/dpower = alpha dL/dalpha = (o G) c
    assert np.isclose(g[5], c * G, rtol=1e-6)        # dL/do
    assert np.isclose(g[2], -0.5 * 4.0 * dP, rtol=1e-6)          # dA = -0.5 dx^2 dP
    assert np.isclose(g[0], -(A * -2.0) * dP, rtol=1e-6)         # du = -(A dx + B dy) dP
    assert np.isclose(g[1], -(0.3 * -2.0) * dP, rtol=1e-6)       # dv = -(C dy + B dx) dP
    assert abs(g[3]) < 1e-12 and abs(g[4]) < 1e-12               # dB ~ dx dy = 0, dC ~ dy^2 = 0
    assert np.isclose(g[6], o * G, rtol=1e-6)


def test_clamped_alpha_passes_no_gradient_to_opacity_or_shape(ho):
    proj = _one(3.0, 2.0, 0.5, 0.0, 0.5, 0.999, (0.5, 0.5, 0.5))   # o exp(0) = 0.999 > 0.99 at the centre
    lr, rg = _lists(16, 16, 1)
    gc = np.zeros((16, 16, 3), np.float32)
    gc[2, 3] = 1.0
    g = ho.stage_raster_backward(16, 16, proj, lr, rg, gc, np.zeros((16, 16), np.float32))[0]
    assert np.abs(g[:6]).max() == 0.0
    assert np.allclose(g[6:9], 0.99, rtol=1e-6)                    # alpha T = 0.99 (binary32 constant)


def _torch_blend_grads(proj, list_rank, ranges, W, H, gc, gt):
    """The same blend written with torch float64 ops; decisions taken on detached values; autograd does the rest."""
    import torch
    P = torch.tensor(proj.astype(np.float64), requires_grad=True)
    gx = (W + 15) // 16
    loss = torch.zeros((), dtype=torch.float64)
    n_blend = np.zeros((H, W), np.int64)
    for py in range(H):
        for px in range(W):
            t = (py // 16) * gx + px // 16
            T = torch.ones((), dtype=torch.float64)
            Cc = torch.zeros(3, dtype=torch.float64)
            for q in range(int(ranges[t, 0]), int(ranges[t, 1])):
                g = P[int(list_rank[q])]
                dx, dy = g[0] - px, g[1] - py
                power = -0.5 * (g[3] * dx * dx + g[5] * dy * dy) - g[4] * dx * dy
                if power.item() > 0:
                    continue
                alpha = torch.clamp(g[6] * torch.exp(power), max=0.99)
                if alpha.item() < 1.0 / 255.0:
                    continue
                Tn = T * (1 - alpha)
                if Tn.item() < 1e-4:
                    break
                Cc = Cc + g[7:10] * alpha * T
                T = Tn
                n_blend[py, px] += 1
            loss = loss + (Cc * torch.tensor(gc[py, px].astype(np.float64))).sum() + T * float(gt[py, px])
    loss.backward()
    G = P.grad.numpy()
    return np.concatenate([G[:, 0:2], G[:, 3:10]], axis=1), n_blend


@pytest.mark.parametrize("seed,scale_mean", [(7, -2.5), (21, -1.5)])
def test_against_torch_autograd(ho, synth, seed, scale_mean):
    s = synth.tiny_scene(n=40, W=24, H=20, seed=seed, scale_mean=scale_mean)
    r = ho.render(ho.OracleScene(s), s.cameras[0])
    W, H = r["W"], r["H"]
    rng = np.random.default_rng(seed)
    gc = rng.normal(0, 1, (H, W, 3)).astype(np.float32)
    gt = rng.normal(0, 1, (H, W)).astype(np.float32)
    want, nb = _torch_blend_grads(r["proj"], r["list_rank"], r["ranges"], W, H, gc, gt)
    assert (nb == r["n_blend"]).all()          # float64 decisions = the oracle's binary32 decisions on this scene
    assert nb.max() >= 3                       # several layers deep somewhere: the suffix term is exercised
    got = ho.stage_raster_backward(W, H, r["proj"], r["list_rank"], r["ranges"], gc, gt)
    scale = np.abs(want).max(axis=0)
    assert (scale > 0).all()
    assert (np.abs(got - want) <= 2e-5 * scale + 1e-5 * np.abs(want)).all(), np.abs(got - want).max(axis=0) / scale


def test_against_finite_differences_of_the_forward_stage(ho, synth):
    # colour is linear in C_fg and T does not depend on it: central differences of the oracle's own forward are exact
    # up to binary32 rounding; opacity with a small step
    s = synth.tiny_scene(n=30, W=20, H=18, seed=3, scale_mean=-2.0)
    r = ho.render(ho.OracleScene(s), s.cameras[0])
    W, H = r["W"], r["H"]
    rng = np.random.default_rng(1)
    gc = rng.normal(0, 1, (H, W, 3)).astype(np.float32)
    gt = rng.normal(0, 1, (H, W)).astype(np.float32)
    got = ho.stage_raster_backward(W, H, r["proj"], r["list_rank"], r["ranges"], gc, gt)

    def loss(proj):
        f = ho.stage_raster(W, H, proj, r["list_rank"], r["ranges"])
        return float((f["cfg"].astype(np.float64) * gc).sum() + (f["T"].astype(np.float64) * gt).sum()), f["n_blend"]

    checked = 0
    for g in np.argsort(-np.abs(got[:, 5]))[:6]:
        for col, k, eps in ((7, 6, 0.25), (9, 8, 0.25), (6, 5, 2e-3)):
            pp, pm = r["proj"].copy(), r["proj"].copy()
            pp[g, col] += eps
            pm[g, col] -= eps
            (lp, nbp), (lm, nbm) = loss(pp), loss(pm)
            if not ((nbp == r["n_blend"]).all() and (nbm == r["n_blend"]).all()):
                continue                        # a decision flipped inside the step: not a derivative of the frozen set
            fd = (lp - lm) / (2 * eps)
            assert abs(fd - got[g, k]) <= 2e-3 * max(1.0, abs(got[g, k])), (g, col, fd, got[g, k])
            checked += 1
    assert checked >= 10
