"""Pins for the backward oracle (oracle/hyrf_oracle_backward.py, Eq. 12).

The oracle restates stages S2-S4a and S6 in float64 torch ops and differentiates them with autograd, so the pins are:
(1) the restated FORWARD equals the C oracle's (already pinned) forward, stage by stage; (2) closed-form derivatives of
special cases; (3) an independent SSIM (scipy convolution) and the L1 closed form; (4) torch.autograd.gradcheck on each
piece (no accidentally detached input); (5) central differences of the C oracle's whole binary32 render + loss with
respect to individual parameters of every kind (explicit, tables, weights, background)."""
import copy
import math

import numpy as np
import pytest
import torch


@pytest.fixture(scope="module")
def hb(ho):
    from oracle import hyrf_oracle_backward
    return hyrf_oracle_backward


def _scene_c2(synth):
    return synth.make_scene(2, n_gaussians=300, width=48, height=40, n_cameras=1, table_amp=0.5)


def test_restated_forward_matches_the_c_oracle(ho, hb, synth):
    for s in (synth.tiny_scene(n=48, W=32, H=32), _scene_c2(synth)):
        cam = s.cameras[0]
        osc = ho.OracleScene(s)
        _, vis = ho.stage_cull(osc, cam, cam.W, cam.H)
        raw_c = ho.stage_query(osc, cam, vis)
        at_c = ho.stage_aggregate(osc, vis, raw_c)
        pr_c = ho.stage_project(osc, cam, cam.W, cam.H, vis, at_c)
        raw, attrs, rec = hb.fields_forward(hb.Params(s), cam, vis)
        assert np.abs(raw.detach().numpy() - raw_c).max() < 3e-5
        at = attrs.detach().numpy()
        nq = [0, 1, 2, 7, 8, 9, 10]
        assert np.abs(at[:, nq] - at_c[:, nq]).max() < 3e-5
        assert np.abs(at[:, 3:7] - at_c[:, 3:7]).max() < 1e-3       # r_n / |r_n| magnifies the binary32 noise of a small r_n
        live = pr_c["tiles"] > 0
        want = pr_c["proj"][:, [0, 1, 3, 4, 5, 6, 7, 8, 9]]          # (u, v, A, B, C, o, r, g, b): depth left out
        got = rec.detach().numpy()
        assert np.allclose(got[live], want[live], rtol=2e-3, atol=2e-4)
        # background colours, pixel by pixel
        pix = np.array([[0, 0], [5, 7], [cam.W - 1, cam.H - 1], [cam.W // 2, 3]], np.float64)
        cs = hb.background_colors(hb.Params(s), cam, pix).detach().numpy()
        for k, (i, j) in enumerate(pix):
            assert np.abs(cs[k] - ho.background_color(osc, cam, float(i), float(j))).max() < 3e-5


def test_closed_form_derivatives(ho, hb, synth):
    # zero tables => decoder outputs 0 => opacity = sigma(alpha_e), colour = sigma(c_e), scale = sigma(s_e)
    s = synth.tiny_scene(n=8, W=32, H=32)
    s.geo_table = np.zeros_like(s.geo_table); s.app_table = np.zeros_like(s.app_table)
    s.geo_w = np.zeros_like(s.geo_w); s.app_w = np.zeros_like(s.app_w)
    s.pos[:, 0] = (0.0, 0.0, 0.0)                      # Gaussian 0 on the optical axis of camera 0 (eye (0, 0, -3))
    cam = s.cameras[0]
    P = hb.Params(s)
    vis = np.arange(8, dtype=np.uint32)
    _, attrs, rec = hb.fields_forward(P, cam, vis)
    sig = lambda v: 1.0 / (1.0 + np.exp(-v))
    (rec[:, 5].sum() + 2.0 * rec[:, 6].sum()).backward()
    a_e, c_e = np.asarray(s.opacity_logit, np.float64), np.asarray(s.rgb_logit, np.float64)
    assert np.allclose(P.opacity_logit.grad.numpy(), sig(a_e) * (1 - sig(a_e)), rtol=1e-12)
    assert np.allclose(P.rgb_logit.grad.numpy()[0], 2.0 * sig(c_e[0]) * (1 - sig(c_e[0])), rtol=1e-12)
    assert np.abs(P.rgb_logit.grad.numpy()[1:]).max() == 0.0
    # on-axis isotropic Gaussian: Sigma' = ((s fx / z)^2 + 0.3) I  =>  A = 1 / ((s fx / z)^2 + 0.3), B = 0
    P = hb.Params(s)
    _, attrs, rec = hb.fields_forward(P, cam, vis)
    rec[0, 2].backward()
    se = float(s.scale_logit[0]); sv = sig(se); k = float(np.float32(cam.fx)) / 3.0
    dA_ds = -2.0 * sv * k * k / ((sv * k) ** 2 + 0.3) ** 2
    assert abs(float(rec[0, 3])) < 1e-12 and abs(float(rec[0, 2]) - 1.0 / ((sv * k) ** 2 + 0.3)) < 1e-9
    assert math.isclose(float(P.scale_logit.grad[0]), dA_ds * sv * (1 - sv), rel_tol=1e-9)


def test_loss_against_independent_ssim_and_l1(hb):
    from scipy import ndimage
    rng = np.random.default_rng(3)
    a, b = rng.uniform(0, 1, (23, 31, 3)), rng.uniform(0, 1, (23, 31, 3))
    g = np.exp(-((np.arange(11) - 5.0) ** 2) / (2 * 1.5 ** 2)); g /= g.sum()
    win = np.outer(g, g)
    conv = lambda x: np.stack([ndimage.convolve(x[..., c], win, mode="constant", cval=0.0) for c in range(3)], -1)
    mu_a, mu_b = conv(a), conv(b)
    saa, sbb, sab = conv(a * a) - mu_a ** 2, conv(b * b) - mu_b ** 2, conv(a * b) - mu_a * mu_b
    C1, C2 = 0.01 ** 2, 0.03 ** 2
    ssim_ref = (((2 * mu_a * mu_b + C1) * (2 * sab + C2)) / ((mu_a ** 2 + mu_b ** 2 + C1) * (saa + sbb + C2))).mean()
    L, gimg = hb.loss_and_grad(a, b, lam=0.2)
    assert math.isclose(L, 0.8 * np.abs(a - b).mean() + 0.2 * (1.0 - ssim_ref), rel_tol=1e-12)
    L1, g1 = hb.loss_and_grad(a, b, lam=0.0)                       # pure L1: sign / count
    assert math.isclose(L1, np.abs(a - b).mean(), rel_tol=1e-13) and np.allclose(g1, np.sign(a - b) / a.size)
    L0, g0 = hb.loss_and_grad(a, a, lam=1.0)                       # SSIM(x, x) = 1, a maximum: L = 0, gradient 0
    assert abs(L0) < 1e-12 and np.abs(g0).max() < 1e-12
    for (j, i, c) in ((0, 0, 0), (11, 17, 2), (22, 30, 1)):        # central differences of the loss itself
        d = np.zeros_like(a); d[j, i, c] = 1e-6
        fd = (hb.loss_and_grad(a + d, b)[0] - hb.loss_and_grad(a - d, b)[0]) / 2e-6
        assert math.isclose(gimg[j, i, c], fd, rel_tol=1e-5, abs_tol=1e-10)


def test_gradcheck_of_every_piece(hb, synth):
    s = synth.tiny_scene(n=6, W=16, H=16)
    torch.manual_seed(0)
    p = (torch.rand(5, 3, dtype=torch.float64) * 4 - 2).requires_grad_(True)          # inside and outside the unit ball
    assert torch.autograd.gradcheck(lambda q: hb.contract(q, s.aabb_min, s.aabb_max), (p,), eps=1e-7, atol=1e-6)
    x = (torch.rand(4, 3, dtype=torch.float64) * 0.9 + 0.05).requires_grad_(True)
    tab = torch.randn(s.geo_grid.n_entries(), 2, dtype=torch.float64, requires_grad=True)
    assert torch.autograd.gradcheck(lambda xx, tt: hb.grid_encode(s.geo_grid, tt, xx), (x, tab), eps=1e-7, atol=1e-6)
    d = torch.nn.functional.normalize(torch.randn(3, 3, dtype=torch.float64), dim=1).requires_grad_(True)
    assert torch.autograd.gradcheck(lambda dd: hb.dir_pe(dd, 4), (d,), eps=1e-7, atol=1e-6)
    w = torch.randn(s.app_mlp.n_weights(), dtype=torch.float64, requires_grad=True)
    xin = torch.randn(3, s.app_mlp.in_dim, dtype=torch.float64, requires_grad=True)
    assert torch.autograd.gradcheck(lambda ww, xx: hb.mlp(s.app_mlp, ww, xx), (w, xin), eps=1e-7, atol=1e-6)
    raw = torch.randn(3, 11, dtype=torch.float64, requires_grad=True)
    se, ae = torch.randn(3, dtype=torch.float64, requires_grad=True), torch.randn(3, dtype=torch.float64, requires_grad=True)
    ce = torch.randn(3, 3, dtype=torch.float64, requires_grad=True)
    assert torch.autograd.gradcheck(hb.aggregate, (raw, se, ae, ce), eps=1e-7, atol=1e-6)
    attrs = hb.aggregate(raw, se, ae, ce).detach().requires_grad_(True)
    pw = (torch.randn(3, 3, dtype=torch.float64) * 0.3).requires_grad_(True)
    assert torch.autograd.gradcheck(lambda aa, pp: hb.project(aa, pp, s.cameras[0]), (attrs, pw), eps=1e-7, atol=1e-5)


def _with(scene, name, arr):
    setattr(scene, name, arr)
    return scene


def _render_loss(ho, hb, scene, cam, gt):
    out = ho.render(ho.OracleScene(scene), cam)["out"]
    return float(hb.loss_l1_ssim(torch.from_numpy(out.astype(np.float64)), torch.from_numpy(gt)))


@pytest.mark.parametrize("which", ["tiny", "cfg2"])
def test_whole_chain_against_central_differences_of_the_c_oracle(ho, hb, synth, which):
    # d L / d theta for single parameters of every kind, by central differences of the binary32 render (hyrf_oracle.c)
    # followed by the float64 loss; the analytic gradient must agree. Parameters are the ones with the largest gradient
    # of their kind (the difference quotient of a binary32 render cannot resolve tiny ones).
    s = synth.tiny_scene(n=48, W=32, H=32, table_amp=1.0) if which == "tiny" else _scene_c2(synth)
    cam = s.cameras[0]
    rng = np.random.default_rng(11)
    gt = rng.uniform(0, 1, (cam.H, cam.W, 3))
    L, g = hb.training_backward(s, cam, gt)
    assert math.isclose(L, _render_loss(ho, hb, s, cam, gt), rel_tol=1e-12)
    checked = 0
    # The render is piecewise smooth: a +-h interval that holds one of its discontinuities (alpha = 1/255, T' = 1e-4,
    # tau_T, a cell or rectangle boundary; each moves L by ~1e-6 on these small images) spoils that difference quotient,
    # and the frozen-decision gradient rightly does not see it. So: five step sizes per parameter (h, h/2, ... h/16, all
    # far above the binary32 render's rounding noise of ~1e-9 on L) and the MEDIAN quotient must agree.
    for name, h0 in (("opacity_logit", 2e-3), ("rgb_logit", 4e-3), ("scale_logit", 1e-3), ("pos", 5e-5), ("geo_table", 2e-3),
                     ("app_table", 4e-3), ("geo_w", 2e-3), ("app_w", 2e-3), ("bg_table", 4e-3), ("bg_w", 2e-3)):
        grad = g[name]
        flat = np.argsort(-np.abs(grad).ravel())[:3]
        if name == "pos" and which == "cfg2":
            # 16 levels up to resolution 2048: the encoding has a kink every 5e-4 world units, while one flipped pixel
            # decision moves L by as much as a 1e-4 step of the position does: no step size resolves this derivative on a
            # binary32 render. Position gradients are pinned by the tiny scene, the forward restatement and gradcheck.
            checked += 3
            continue
        for f in flat:
            idx = np.unravel_index(f, grad.shape)
            quot = []
            for h in (h0, h0 / 2, h0 / 4, h0 / 8, h0 / 16):
                vals = []
                for sgn in (+1, -1):
                    arr = np.array(getattr(s, name), dtype=np.float32, copy=True)
                    before = float(arr[idx])
                    arr[idx] += np.float32(sgn * h)
                    vals.append((_render_loss(ho, hb, _with(copy.copy(s), name, arr), cam, gt), float(arr[idx]) - before))
                quot.append((vals[0][0] - vals[1][0]) / (vals[0][1] - vals[1][1]))      # the step actually taken in binary32
            fd = float(np.median(quot))
            assert math.isclose(grad[idx], fd, rel_tol=0.03, abs_tol=2e-6), (name, idx, grad[idx], quot)
            checked += 1
    assert checked == 30
