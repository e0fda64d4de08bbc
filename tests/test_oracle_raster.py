"""Pins for the splatting half of the oracle (DESIGN.md §2 D8-D11): closed-form EWA Jacobian (I3), list
properties, transmittance / weight invariants (I4), brute force vs tiled on tiny scenes (I5), ray-sphere
and compositing pins (Eq. 1, 10-11, 15-18)."""
import math

import numpy as np
import pytest


def _quat_to_R(q):
    w, x, y, z = q
    return np.array([[1 - 2 * (y * y + z * z), 2 * (x * y - w * z), 2 * (x * z + w * y)],
                     [2 * (x * y + w * z), 1 - 2 * (x * x + z * z), 2 * (y * z - w * x)],
                     [2 * (x * z - w * y), 2 * (y * z + w * x), 1 - 2 * (x * x + y * y)]])


def _attrs(s3, q, op=0.8, rgb=(0.2, 0.5, 0.9)):
    return np.array(list(s3) + list(q) + [op] + list(rgb), np.float32)


def test_I3_projected_covariance_matches_closed_form_jacobian(ho, synth):
    rng = np.random.default_rng(11)
    cam = synth.look_at(np.array([1.5, -0.8, 2.2]), 320, 200)
    Rc = cam.R.astype(np.float64)
    for _ in range(200):
        s3 = np.exp(rng.uniform(-5, -1, 3))
        q = rng.normal(size=4); q /= np.linalg.norm(q)
        p = rng.uniform(-1, 1, 3)
        pc = Rc @ p + cam.t.astype(np.float64)
        if pc[2] < 0.3:
            continue
        at = _attrs(s3, q)
        r = ho.project(at, pc.astype(np.float32), cam, 320, 200)
        s32, q32, pc32 = at[0:3].astype(np.float64), at[3:7].astype(np.float64), pc.astype(np.float32).astype(np.float64)
        M = _quat_to_R(q32)
        Sigma = M @ np.diag(s32 ** 2) @ M.T
        X, Y, Z = pc32
        J = np.array([[cam.fx / Z, 0, -cam.fx * X / Z ** 2], [0, cam.fy / Z, -cam.fy * Y / Z ** 2]])
        cov = J @ Rc @ Sigma @ Rc.T @ J.T + 0.3 * np.eye(2)
        assert np.allclose(r["cov"], [cov[0, 0], cov[0, 1], cov[1, 1]], rtol=2e-4, atol=2e-5)
        A, B, C = r["proj"][3:6].astype(np.float64)
        conic = np.array([[A, B], [B, C]])
        assert np.allclose(conic @ cov, np.eye(2), atol=2e-3)                  # conic = cov^-1
        lam_max = np.linalg.eigvalsh(cov)[-1]
        assert r["radius"] >= 3 * math.sqrt(lam_max) - 1e-3 and r["radius"] == math.ceil(r["radius"])
        assert np.allclose(r["proj"][0:2], [cam.fx * X / Z + cam.cx, cam.fy * Y / Z + cam.cy], atol=1e-3)
        assert r["proj"][2] == np.float32(pc[2])                               # depth = camera z


def test_on_axis_isotropic_case_and_zero_quaternion(ho, synth):
    cam = synth.Camera(R=np.eye(3, dtype=np.float32), t=np.zeros(3, np.float32), fx=200.0, fy=200.0, cx=99.5,
                       cy=99.5, W=200, H=200)
    s, z = 0.05, 4.0
    r = ho.project(_attrs([s, s, s], [1, 0, 0, 0]), [0, 0, z], cam, 200, 200)
    v = (s * 200.0 / z) ** 2 + 0.3
    assert np.allclose(r["cov"], [v, 0, v], rtol=1e-6)                          # ((s fx/z)^2 + 0.3) I
    assert np.allclose(r["proj"][3:6], [1 / v, 0, 1 / v], rtol=1e-6)
    assert r["radius"] == math.ceil(3 * math.sqrt(v))
    assert np.allclose(r["proj"][0:2], [99.5, 99.5])
    # rotation does not matter for an isotropic Gaussian
    q = np.array([0.3, -0.5, 0.7, 0.1]); q /= np.linalg.norm(q)
    r2 = ho.project(_attrs([s, s, s], q), [0, 0, z], cam, 200, 200)
    assert np.allclose(r2["cov"], r["cov"], rtol=1e-5, atol=1e-5)
    # zero quaternion (the "w/o Neural" fallback) behaves as the identity rotation
    r3 = ho.project(_attrs([s, s, s], [0, 0, 0, 0]), [0, 0, z], cam, 200, 200)
    assert (r3["cov"] == r["cov"]).all()


def test_tile_rect_rule(ho, synth):
    cam = synth.Camera(R=np.eye(3, dtype=np.float32), t=np.zeros(3, np.float32), fx=100.0, fy=100.0, cx=0.0, cy=0.0,
                       W=100, H=70)                                                # 7 x 5 tiles
    # tiny Gaussian at pixel (40, 24): lambda = 0.3 + sqrt(max(0.1, 0)) (the 0.1 floor) -> radius = ceil(3 sqrt(0.616)) = 3
    # -> x in [37,43] -> tile column 2, y in [21,27] -> tile row 1
    r = ho.project(_attrs([1e-4] * 3, [1, 0, 0, 0]), [0.4, 0.24, 1.0], cam, 100, 70)
    assert r["radius"] == 3.0
    assert r["rect"].tolist() == [2, 3, 1, 2] and r["tiles"] == 1
    # centre on a tile corner (48, 32): touches 4 tiles
    r = ho.project(_attrs([1e-4] * 3, [1, 0, 0, 0]), [0.48, 0.32, 1.0], cam, 100, 70)
    assert r["rect"].tolist() == [2, 4, 1, 3] and r["tiles"] == 4
    # partially off the left/top edge: clamped at 0
    r = ho.project(_attrs([1e-4] * 3, [1, 0, 0, 0]), [0.0, 0.0, 1.0], cam, 100, 70)
    assert r["rect"].tolist() == [0, 1, 0, 1]
    # entirely off-screen to the right: x0 = x1 = grid -> dropped
    r = ho.project(_attrs([1e-4] * 3, [1, 0, 0, 0]), [2.0, 0.3, 1.0], cam, 100, 70)
    assert r["tiles"] == 0
    # large Gaussian covers the whole grid, never more
    r = ho.project(_attrs([5.0] * 3, [1, 0, 0, 0]), [0.5, 0.3, 1.0], cam, 100, 70)
    assert r["rect"].tolist() == [0, 7, 0, 5] and r["tiles"] == 35


def _render_tiny(ho, synth, **kw):
    s = synth.tiny_scene(**kw)
    osc = ho.OracleScene(s)
    return s, osc, [ho.render(osc, c) for c in s.cameras]


def test_O8_list_properties(ho, synth):
    s, osc, frames = _render_tiny(ho, synth, n=64, W=48, H=40)
    for r in frames:
        gx = (r["W"] + 15) // 16
        assert r["D"] == int(r["tiles"].sum()) == len(r["list_id"])
        depth_bits = r["proj"][:, 2].view(np.uint32)
        covered = 0
        for t, (a, b) in enumerate(r["ranges"]):
            ids, rk = r["list_id"][a:b], r["list_rank"][a:b]
            assert len(set(ids.tolist())) == len(ids)                               # each (tile, id) at most once
            keys = list(zip(depth_bits[rk].tolist(), ids.tolist()))
            assert keys == sorted(keys)                                              # (depth bits, id) ascending
            tx, ty = t % gx, t // gx
            member = [(rc[0] <= tx < rc[1]) and (rc[2] <= ty < rc[3]) and tl > 0 for rc, tl in zip(r["rect"], r["tiles"])]
            assert sorted(ids.tolist()) == sorted(r["vis_idx"][np.nonzero(member)[0]].tolist())   # iff rect covers tile
            covered += b - a
        assert covered == r["D"]
        assert (r["vis_idx"][r["list_rank"]] == r["list_id"]).all()


def test_depth_ties_break_by_id(ho, synth):
    # two Gaussians at identical positions (equal depth bits) -> ascending id inside every tile (reading A16)
    s = synth.tiny_scene(n=6)
    s.pos[:, 4] = s.pos[:, 1]
    s.pos[:, 2] = s.pos[:, 1]
    r = ho.render(ho.OracleScene(s), s.cameras[0])
    for a, b in r["ranges"]:
        ids = r["list_id"][a:b].tolist()
        trio = [i for i in ids if i in (1, 2, 4)]
        assert trio == sorted(trio)


def test_I4_transmittance_and_weights(ho, synth):
    s, osc, frames = _render_tiny(ho, synth, n=64, W=32, H=32, scale_mean=-2.0)
    for r in frames:
        T = r["T"]
        assert (T >= 0).all() and (T <= 1).all()
        assert np.allclose(r["wsum"] + T, 1.0, atol=2e-6)                            # sum w_i + T_final = 1
        assert (r["n_blend"] <= r["n_eval"]).all() and r["n_blend"].max() > 3
        assert (T[r["n_blend"] == 0] == 1.0).all()
        assert T.min() < 0.5                                                         # something is actually blended


def test_transmittance_monotone_along_list(ho, synth):
    # recompute the prefix transmittances of a few pixels from pair_alpha: non-increasing, inside [0,1]
    s, osc, frames = _render_tiny(ho, synth, n=64, W=32, H=32, scale_mean=-2.0)
    r = frames[0]
    for (px, py) in [(5, 7), (16, 16), (30, 2), (12, 25)]:
        a, b = r["ranges"][(py // 16) * 2 + px // 16]
        T, Ts = np.float32(1), []
        for q in range(a, b):
            al, skipped = ho.pair_alpha(r["proj"][r["list_rank"][q]], px, py)
            if skipped or np.float32(al) < np.float32(1 / 255):
                continue
            Tn = np.float32(T * (np.float32(1) - np.float32(al)))
            if Tn < np.float32(1e-4):
                break
            T = Tn
            Ts.append(float(T))
        assert all(x >= y for x, y in zip([1.0] + Ts, Ts)) and all(0 <= x <= 1 for x in Ts)
        assert np.float32(T) == r["T"][py, px]


def test_constant_colour_scene_gives_constant_image(ho, synth):
    # all Gaussian colours = k and background = k  ->  image = k  (weights + residual sum to 1)
    s = synth.tiny_scene(n=64, W=32, H=32, scale_mean=-2.0)
    k = 0.3
    logit = math.log(k / (1 - k))
    s.rgb_logit[:] = logit
    s.app_w = np.zeros_like(s.app_w)                # c_n = 0 -> c = sigma(c_e) = k
    s.bg_w = np.zeros_like(s.bg_w)                  # c_s = sigma(0) = 0.5
    s.tau_T = 0.0
    r = ho.render(ho.OracleScene(s), s.cameras[0])
    fg_expect = k * (1 - r["T"])
    assert np.allclose(r["cfg"], fg_expect[..., None], atol=3e-6)
    assert np.allclose(r["out"], (fg_expect + 0.5 * r["T"])[..., None], atol=3e-6)


def test_single_opaque_gaussian_at_pixel_centre(ho, synth):
    cam = synth.Camera(R=np.eye(3, dtype=np.float32), t=np.zeros(3, np.float32), fx=64.0, fy=64.0, cx=15.5, cy=15.5,
                       W=32, H=32)
    for op, expect in [(0.6, 0.6), (0.999, 0.99)]:                                    # alpha = min(0.99, o)
        proj = np.array([[8.0, 9.0, 2.0, 0.5, 0.0, 0.5, op, 1.0, 0.5, 0.25]], np.float32)
        ranges = np.zeros((4, 2), np.uint32); ranges[0] = [0, 1]
        rs = ho.stage_raster(32, 32, proj, np.zeros(1, np.uint32), ranges)
        assert abs(rs["T"][9, 8] - (1 - expect)) < 1e-7
        assert np.allclose(rs["cfg"][9, 8], np.array([1.0, 0.5, 0.25]) * expect, atol=1e-7)
        # Gaussian falloff: alpha(dx) = o exp(-0.5 A dx^2)
        assert abs((1 - rs["T"][9, 10]) - min(0.99, op * math.exp(-0.5 * 0.5 * 4))) < 1e-6
        assert (rs["T"][16:, :] == 1).all() and (rs["T"][:, 16:] == 1).all()          # other tiles untouched


def test_stop_rule_and_skip_rule(ho):
    # four layers of alpha 0.95: T = 0.05, 0.0025, 1.25e-4, then T' = 6.25e-6 < 1e-4 -> stop BEFORE blending the 4th
    base = [8.0, 8.0, 1.0, 0.01, 0.0, 0.01, 0.95]
    proj = np.array([base + [1, 0, 0], base + [0, 1, 0], base + [0, 0, 1], base + [1, 1, 1]], np.float32)
    proj[:, 2] = [1, 2, 3, 4]
    ranges = np.array([[0, 4]], np.uint32)
    rs = ho.stage_raster(16, 16, proj, np.arange(4, dtype=np.uint32), ranges)
    assert rs["n_blend"][8, 8] == 3 and abs(rs["T"][8, 8] - 1.25e-4) < 1e-9
    assert np.allclose(rs["cfg"][8, 8], [0.95, 0.95 * 0.05, 0.95 * 0.0025], atol=1e-7)
    # alpha below 1/255 is skipped: opacity 0.0039 < 1/255 = 0.00392
    proj2 = np.array([[8.0, 8.0, 1.0, 0.01, 0.0, 0.01, 0.0039, 1, 1, 1]], np.float32)
    rs2 = ho.stage_raster(16, 16, proj2, np.zeros(1, np.uint32), np.array([[0, 1]], np.uint32))
    assert rs2["T"][8, 8] == 1.0 and rs2["n_blend"][8, 8] == 0 and rs2["n_eval"][8, 8] == 1


def test_pair_alpha_closed_form(ho):
    rng = np.random.default_rng(12)
    for _ in range(300):
        a, c = rng.uniform(0.4, 50, 2); b = rng.uniform(-0.9, 0.9) * math.sqrt(a * c)
        det = a * c - b * b
        A, B, C = c / det, -b / det, a / det
        u, v, op = rng.uniform(0, 32), rng.uniform(0, 32), rng.uniform(0.01, 1)
        i, j = rng.integers(0, 32, 2)
        proj = np.array([u, v, 1, A, B, C, op, 0, 0, 0], np.float32)
        al, skipped = ho.pair_alpha(proj, float(i), float(j))
        p32 = proj.astype(np.float64)
        dx, dy = p32[0] - i, p32[1] - j
        power = -0.5 * (p32[3] * dx * dx + p32[5] * dy * dy) - p32[4] * dx * dy
        assert not skipped
        assert abs(al - min(0.99, p32[6] * math.exp(power))) < 1e-6


@pytest.mark.parametrize("seed", [7, 8, 9])
def test_I5_brute_force_equals_tiled(ho, synth, seed):
    """Tiny scene: every pixel blends ALL Gaussians sorted globally by (depth bits, id), restricted by the rect
    membership rule of SURVEY H3; must equal the tiled result bit for bit."""
    s = synth.tiny_scene(n=56, W=32, H=32, seed=seed, scale_mean=-2.2)
    osc = ho.OracleScene(s)
    for cam in s.cameras:
        r = ho.render(osc, cam)
        V = len(r["vis_idx"])
        depth_bits = r["proj"][:, 2].view(np.uint32)
        order = sorted(range(V), key=lambda j: (int(depth_bits[j]), int(r["vis_idx"][j])))
        one255, stop = np.float32(1 / 255), np.float32(1e-4)
        for py in range(0, 32):
            for px in range(0, 32):
                tx, ty = px // 16, py // 16
                T = np.float32(1); Cc = np.zeros(3, np.float32)
                for j in order:
                    rc = r["rect"][j]
                    if r["tiles"][j] == 0 or not (rc[0] <= tx < rc[1] and rc[2] <= ty < rc[3]):
                        continue
                    al, skipped = ho.pair_alpha(r["proj"][j], px, py)
                    al = np.float32(al)
                    if skipped or al < one255:
                        continue
                    Tn = np.float32(T * np.float32(np.float32(1) - al))
                    if Tn < stop:
                        break
                    wgt = np.float32(al * T)
                    # fma(c, w, C): fp64 product+sum of fp32 values rounded once equals fmaf here except on
                    # double-rounding ties; compare colour at 1 ulp, T and decisions exactly
                    Cc = (Cc.astype(np.float64) + r["proj"][j, 7:10].astype(np.float64) * float(wgt)).astype(np.float32)
                    T = Tn
                assert T == r["T"][py, px]
                assert np.allclose(Cc, r["cfg"][py, px], rtol=0, atol=3e-7)


def test_brute_force_fp64_independent_of_tiling(ho, synth):
    # the same check in fp64 numpy without any oracle arithmetic: Eq. 1 over the rect-membership set
    s = synth.tiny_scene(n=56, W=32, H=32, seed=21, scale_mean=-2.2)
    r = ho.render(ho.OracleScene(s), s.cameras[0])
    P = r["proj"].astype(np.float64)
    depth_bits = r["proj"][:, 2].view(np.uint32)
    order = np.lexsort((r["vis_idx"], depth_bits))
    bad = 0
    for py in range(32):
        for px in range(32):
            T, Cc = 1.0, np.zeros(3)
            for j in order:
                rc = r["rect"][j]
                if r["tiles"][j] == 0 or not (rc[0] <= px // 16 < rc[1] and rc[2] <= py // 16 < rc[3]):
                    continue
                dx, dy = P[j, 0] - px, P[j, 1] - py
                power = -0.5 * (P[j, 3] * dx * dx + P[j, 5] * dy * dy) - P[j, 4] * dx * dy
                if power > 0:
                    continue
                al = min(0.99, P[j, 6] * math.exp(power))
                if al < 1 / 255:
                    continue
                if T * (1 - al) < 1e-4:
                    break
                Cc += P[j, 7:10] * al * T
                T *= 1 - al
            fragile = r["m_alpha"][py, px] < 1e-6 or r["m_stop"][py, px] < 1e-3
            if not fragile:
                assert abs(T - r["T"][py, px]) < 1e-5 and np.allclose(Cc, r["cfg"][py, px], atol=1e-5)
            bad += fragile
    assert bad < 10
