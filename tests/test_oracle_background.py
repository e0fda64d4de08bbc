"""Pins for stage 6 (PAPER.md:124-134 Eq. 10-11, :360-378 Eq. 15-18) and whole-pass sanity of the oracle."""
import math

import numpy as np


def test_ray_sphere_hits_the_sphere_in_front(ho, synth):
    rng = np.random.default_rng(13)
    for eye in ([0.5, 0.2, -3.0], [30.0, -20.0, 60.0], [0.01, 0.0, 0.0]):
        cam = synth.look_at(np.array(eye), 64, 48)
        o = ho.camera_center(cam).astype(np.float64)
        for _ in range(50):
            i, j = rng.uniform(0, 63), rng.uniform(0, 47)
            d, ps = ho.ray_sphere(cam, float(i), float(j), 100.0)
            assert abs(np.linalg.norm(d) - 1) < 1e-6
            assert abs(np.linalg.norm(ps.astype(np.float64)) - 100.0) < 2e-3          # |p_s| = r  (1e-5 relative)
            t = (ps.astype(np.float64) - o) @ d.astype(np.float64)
            assert t > 0                                                               # the positive root
            assert np.allclose(o + t * d, ps, atol=1e-3)
            # direction agrees with the pinhole model: R d is parallel to ((i-cx)/fx, (j-cy)/fy, 1)
            dc = cam.R.astype(np.float64) @ d.astype(np.float64)
            assert np.allclose(dc[:2] / dc[2], [(i - cam.cx) / cam.fx, (j - cam.cy) / cam.fy], atol=1e-5)


def test_ray_sphere_camera_at_origin(ho, synth):
    cam = synth.Camera(R=np.eye(3, dtype=np.float32), t=np.zeros(3, np.float32), fx=50.0, fy=50.0, cx=31.5, cy=23.5,
                       W=64, H=48)
    for (i, j) in [(0, 0), (31.5, 23.5), (63, 47), (10, 40)]:
        d, ps = ho.ray_sphere(cam, float(i), float(j), 100.0)
        assert np.allclose(ps, 100.0 * d, atol=1e-4)                                   # o = 0 -> p_s = r d


def test_discriminant_positive_inside_sphere(ho, synth):
    # Eq. 18 with |o| < r: disc = B^2 - 4C > 0 always -> finite hit for cameras close to the sphere
    cam = synth.look_at(np.array([0.0, 0.0, -99.9]), 32, 32)
    for (i, j) in [(0, 0), (16, 16), (31, 31)]:
        d, ps = ho.ray_sphere(cam, float(i), float(j), 100.0)
        assert np.isfinite(ps).all() and abs(np.linalg.norm(ps.astype(np.float64)) - 100) < 5e-3


def test_tau_zero_composites_every_pixel_with_T_positive_and_additivity(ho, synth):
    s = synth.tiny_scene(n=48, W=32, H=32, scale_mean=-2.0)
    osc = ho.OracleScene(s)
    cam = s.cameras[0]
    r = ho.render(osc, cam)
    # default tau_T = 0.2: strict T > tau_T (reading A17)
    assert ((r["T"] > np.float32(0.2)) == r["bg_mask"].astype(bool)).all()
    assert 0 < r["bg_mask"].mean() < 1
    off = ~r["bg_mask"].astype(bool)
    assert (r["out"][off] == r["cfg"][off]).all()                                      # C = C_fg where not composited
    s.tau_T = 0.0
    r0 = ho.render(ho.OracleScene(s), cam)
    assert (r0["bg_mask"].astype(bool) == (r0["T"] > 0)).all()
    # Eq. 10-11: C = C_fg + T c_s with c_s the per-pixel background colour
    for (px, py) in [(0, 0), (13, 7), (31, 31), (16, 15)]:
        cs = ho.background_color(osc, cam, float(px), float(py))
        assert (cs > 0).all() and (cs < 1).all()
        expect = r0["cfg"][py, px].astype(np.float64) + float(r0["T"][py, px]) * cs.astype(np.float64)
        assert np.allclose(r0["out"][py, px], expect, atol=1e-6)


def test_background_color_equals_its_parts(ho, synth):
    s = synth.tiny_scene(n=8, table_amp=1.0)
    osc = ho.OracleScene(s)
    cam = s.cameras[1]
    d, ps = ho.ray_sphere(cam, 5.0, 9.0, s.bg_radius)
    x = ho.contract(ps, s.aabb_min, s.aabb_max)
    assert np.abs(x - 0.5).max() > 0.3                                                 # far point -> near the boundary
    f = ho.grid_encode(s.bg_grid, s.bg_table, x)
    raw = ho.mlp_forward(s.bg_mlp, s.bg_w, np.concatenate([f, ho.dir_pe(d)]))
    cs = ho.background_color(osc, cam, 5.0, 9.0)
    assert np.allclose(cs, 1 / (1 + np.exp(-raw.astype(np.float64))), atol=1e-7)


def test_whole_pass_config1_statistics(ho, synth):
    # SURVEY §8 [probe] sizes for cfg 1: V = 4096 (all visible), D ~ 7.7k, ~70% of pixels get background
    s = synth.make_scene(1)
    r = ho.render(ho.OracleScene(s), s.cameras[0])
    assert len(r["vis_idx"]) == 4096
    assert 6000 < r["D"] < 10000
    assert 0.6 < r["bg_mask"].mean() < 0.8
    assert np.isfinite(r["out"]).all() and 0 <= r["out"].min() and r["out"].max() <= 1.0 + 1e-6
    assert np.abs(r["raw"]).max() < 1.5 and np.abs(r["raw"][:, :8]).std() > 1e-3     # weak but non-zero signal (H5)


def test_thread_count_does_not_change_results(ho, synth):
    s = synth.make_scene(2, n_gaussians=3000, width=96, height=64, n_cameras=1)
    osc = ho.OracleScene(s)
    n0 = ho.num_threads()
    ho.set_num_threads(1)
    a = ho.render(osc, s.cameras[0])
    ho.set_num_threads(max(2, n0))
    b = ho.render(osc, s.cameras[0])
    ho.set_num_threads(n0)
    for k in ("mask", "list_id", "out", "T", "raw"):
        assert (a[k] == b[k]).all()


def test_pre_culling_off_changes_only_band_gaussians(ho, synth):
    # PAPER.md:261 "equivalent visual quality": with tol -> inf, extra Gaussians all have centres outside the band
    s = synth.make_scene(3, n_gaussians=5000, width=160, height=96, n_cameras=1)
    cam = s.cameras[0]
    r = ho.render(ho.OracleScene(s), cam)
    s.cull_tol = 1e30
    r2 = ho.render(ho.OracleScene(s), cam)
    extra = np.setdiff1d(r2["vis_idx"], r["vis_idx"])
    assert len(extra) > 0 and set(r["vis_idx"].tolist()) <= set(r2["vis_idx"].tolist())
    lim = 1.1 * cam.W / (2 * cam.fx)
    for i in extra[:200]:
        pc = ho.to_camera(cam, s.pos[:, i])
        assert abs(pc[0]) > lim * pc[2] * (1 - 1e-6) or abs(pc[1]) > 1.1 * cam.H / (2 * cam.fy) * pc[2] * (1 - 1e-6)
    assert np.abs(r2["out"] - r["out"]).mean() < 5e-3
