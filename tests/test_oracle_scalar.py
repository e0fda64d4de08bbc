"""Pins for the oracle's scalar pieces: fp16 conversion, soft exp / sigmoid (DESIGN.md §2 D6), cull (D1),
contraction (D2). Each pin is something other than the oracle's own formula: a library routine (numpy half
casts, math.exp in fp64), a closed form, an invariant or a hand-placed case."""
import math

import numpy as np
import pytest


def test_half_conversion_matches_numpy_exhaustive_decode(ho):
    # every one of the 65536 half bit patterns decodes like numpy's float16 -> float32 (library routine)
    bits = np.arange(65536, dtype=np.uint16)
    ref = bits.view(np.float16).astype(np.float32)
    got = np.array([ho.half_to_float(int(b)) for b in bits[::7]], dtype=np.float32)
    r = ref[::7]
    ok = (got == r) | (np.isnan(got) & np.isnan(r))
    assert ok.all()


def test_float_to_half_matches_numpy_rne(ho):
    rng = np.random.default_rng(0)
    vals = np.concatenate([
        rng.normal(0, 1, 4000), rng.normal(0, 1e-4, 2000), rng.normal(0, 1e-7, 2000), rng.uniform(-70000, 70000, 2000),
        np.array([0.0, -0.0, 65504.0, 65519.9, 65520.0, 1e9, -1e9, 6.1e-5, 5.96e-8, 2.98e-8, 2.9802322e-8, 1e-10]),
        # exact ties between neighbouring halves (must go to even)
        np.array([1.0 + 2.0 ** -11, 1.0 + 3 * 2.0 ** -11, 2048.0 + 1.0, 2048.0 + 3.0]),
    ]).astype(np.float32)
    with np.errstate(over="ignore"):
        ref = vals.astype(np.float16).view(np.uint16)
    got = np.array([ho.float_to_half(float(v)) for v in vals], dtype=np.uint16)
    assert (got == ref).all()


def test_softexp_accuracy_against_fp64(ho):
    xs = np.linspace(-80, 80, 4001).astype(np.float32)
    for x in xs:
        ref = math.exp(float(x))
        got = ho.softexp(float(x))
        assert abs(got - ref) <= 4e-7 * ref, (x, got, ref)
    assert ho.softexp(0.0) == 1.0
    # clamps instead of overflowing / flushing
    assert math.isfinite(ho.softexp(1000.0)) and ho.softexp(-1000.0) > 0.0


def test_sigmoid_closed_form_and_symmetry(ho):
    assert ho.sigmoid(0.0) == 0.5
    for v in np.linspace(-20, 20, 401):
        ref = 1.0 / (1.0 + math.exp(-float(np.float32(v))))
        assert abs(ho.sigmoid(float(v)) - ref) < 2e-7
        assert abs(ho.sigmoid(float(v)) + ho.sigmoid(float(-v)) - 1.0) < 3e-7
    # sigma(-4) = 0.0180 (the regime of the configs' scale logits)
    assert abs(ho.sigmoid(-4.0) - 0.017986) < 1e-6


# ------------------------------------------------------------------------------------------------ D1 cull
class _Scene:
    pass


def _cull_scene(synth, pts, tol=0.1, z_near=0.2):
    s = synth.tiny_scene(n=len(pts))
    s.pos = np.ascontiguousarray(np.asarray(pts, np.float32).T)
    s.cull_tol, s.z_near = tol, z_near
    return s


def test_cull_hand_placed_points(ho, synth):
    # identity camera at the origin looking down +z, fx = fy = 50, 100x100 image -> W/(2fx) = 1 -> limit 1+tol
    cam = synth.Camera(R=np.eye(3, dtype=np.float32), t=np.zeros(3, np.float32), fx=50.0, fy=50.0, cx=49.5, cy=49.5,
                       W=100, H=100)
    lim = float(np.float32(1.0) + np.float32(0.1))           # fp32 (1 + tol)
    pts = [
        (0, 0, 1),            # centre: keep
        (lim * 2, 0, 2),      # exactly on the right plane (x = lim*z, representable product): keep (<=)
        (np.nextafter(np.float32(lim * 2), np.float32(10)), 0, 2),   # one ulp outside: cull
        (-lim * 2, 0, 2),     # exactly on the left plane: keep
        (0, lim * 4, 4),      # exactly on the bottom plane: keep
        (0, -1.2 * 4, 4),     # outside top: cull
        (0, 0, 0.2),          # z == z_near: cull (strict >)
        (0, 0, np.nextafter(np.float32(0.2), np.float32(1))),        # just beyond near: keep
        (0, 0, -1),           # behind: cull
        (1.05, 1.05, 1),      # inside the tolerance band: keep
        (float("nan"), 0, 1), # NaN: cull
    ]
    s = _cull_scene(synth, pts)
    mask, idx = ho.stage_cull(ho.OracleScene(s), cam, 100, 100)
    assert mask.tolist() == [1, 1, 0, 1, 1, 0, 0, 1, 0, 1, 0]
    assert idx.tolist() == [0, 1, 3, 4, 7, 9]


def test_cull_non_square_image_and_anisotropic_focal(ho, synth):
    # every other cull pin has W = H and fx = fy, so a W <-> H or fx <-> fy slip in limx / limy would pass.
    # 160 x 96 image, fx = 50, fy = 100: W/(2 fx) = 1.6, H/(2 fy) = 0.48 (D1: limx = (1 + tol) W / (2 fx),
    # limy = (1 + tol) H / (2 fy), fp32). z = 2 keeps lim * z exact, so "on the plane" is well defined.
    cam = synth.Camera(R=np.eye(3, dtype=np.float32), t=np.zeros(3, np.float32), fx=50.0, fy=100.0, cx=79.5, cy=47.5,
                       W=160, H=96)
    one_tol = np.float32(1.0) + np.float32(0.1)
    limx = one_tol * (np.float32(160.0) / (np.float32(2.0) * np.float32(50.0)))
    limy = one_tol * (np.float32(96.0) / (np.float32(2.0) * np.float32(100.0)))
    assert abs(float(limx) - 1.76) < 1e-6 and abs(float(limy) - 0.528) < 1e-6
    up = lambda v: np.nextafter(np.float32(v), np.float32(1e9))
    pts = [
        (0, limy * 2, 2),            # exactly on the bottom plane: keep
        (0, up(limy * 2), 2),        # one ulp below it: cull
        (0, -limy * 2, 2),           # exactly on the top plane: keep
        (0, -up(limy * 2), 2),       # one ulp above it: cull
        (limx * 2, 0, 2),            # exactly on the right plane: keep
        (up(limx * 2), 0, 2),        # one ulp outside: cull
        (-limx * 2, 0, 2),           # exactly on the left plane: keep
        (1.7 * 2, 0, 2),             # inside limx = 1.76; outside every swapped variant (H/(2fx): 1.056, W/(2fy): 0.88, H/(2fy): 0.528)
        (0, 0.6 * 2, 2),             # outside limy = 0.528; inside every swapped variant (0.88, 1.056, 1.76)
        (1.7 * 2, limy * 2, 2),      # corner of the band: keep
    ]
    s = _cull_scene(synth, pts)
    mask, idx = ho.stage_cull(ho.OracleScene(s), cam, 160, 96)
    assert mask.tolist() == [1, 0, 1, 0, 1, 0, 1, 1, 0, 1]
    assert idx.tolist() == [0, 2, 4, 6, 7, 9]
    # the same through a rotated camera (rows of R permuted: camera x = world y, camera y = world x), so that the
    # limits are tied to the CAMERA axes, not to the world's
    Rp = np.array([[0, 1, 0], [1, 0, 0], [0, 0, 1]], np.float32)
    cam2 = synth.Camera(R=Rp, t=np.zeros(3, np.float32), fx=50.0, fy=100.0, cx=79.5, cy=47.5, W=160, H=96)
    s2 = _cull_scene(synth, [(p[1], p[0], p[2]) for p in pts])
    mask2, _ = ho.stage_cull(ho.OracleScene(s2), cam2, 160, 96)
    assert mask2.tolist() == mask.tolist()


def test_cull_infinite_tolerance_keeps_everything_in_front(ho, synth):
    s = synth.make_scene(1)
    s.cull_tol = 1e30
    cam = s.cameras[0]
    mask, idx = ho.stage_cull(ho.OracleScene(s), cam, cam.W, cam.H)
    z = np.array([ho.to_camera(cam, s.pos[:, i])[2] for i in range(0, s.n, 37)])
    assert (mask[::37].astype(bool) == (z > np.float32(s.z_near))).all()


def test_cull_invariant_under_reordering_and_idx_sorted(ho, synth):
    s = synth.make_scene(3, n_gaussians=20000, n_cameras=3)
    cam = s.cameras[1]
    mask, idx = ho.stage_cull(ho.OracleScene(s), cam, cam.W, cam.H)
    assert 0.3 < mask.mean() < 0.9                      # cfg 3: roughly 40% out of frustum
    assert (np.diff(idx.astype(np.int64)) > 0).all() and (idx == np.nonzero(mask)[0]).all()
    perm = np.random.default_rng(1).permutation(s.n)
    s2 = synth.make_scene(3, n_gaussians=20000, n_cameras=3)
    s2.pos = np.ascontiguousarray(s.pos[:, perm])
    mask2, _ = ho.stage_cull(ho.OracleScene(s2), cam, cam.W, cam.H)
    assert (mask2 == mask[perm]).all()


def test_to_camera_matches_fp64_matrix_product(ho, synth):
    s = synth.make_scene(2, n_gaussians=100)
    for cam in s.cameras:
        R, t = cam.R.astype(np.float64), cam.t.astype(np.float64)
        assert np.allclose(R @ R.T, np.eye(3), atol=1e-6)       # look-at gives a rotation
        for i in range(0, 100, 9):
            p = s.pos[:, i]
            assert np.allclose(ho.to_camera(cam, p), R @ p.astype(np.float64) + t, atol=2e-6)
        o = ho.camera_center(cam)
        assert np.allclose(R @ o.astype(np.float64) + t, 0, atol=2e-6)      # o = -R^T t
        assert abs(np.linalg.norm(o) - 3.0) < 1e-5


# ------------------------------------------------------------------------------------------------ D2 contraction
def test_contract_inside_unit_ball_is_affine(ho):
    amin, amax = [-2, -2, -2], [2, 2, 2]
    for p in ([0, 0, 0], [2, 0, 0], [0, -2, 0], [1, 1, 1], [-0.4, 0.8, 1.2]):
        x = ho.contract(p, amin, amax)
        n = np.linalg.norm(np.array(p) / 2.0)
        if n <= 1:
            assert np.allclose(x, 0.25 * np.array(p) / 2.0 + 0.5, atol=1e-7)
            assert (x >= 0.25 - 1e-7).all() and (x <= 0.75 + 1e-7).all()


def test_contract_range_continuity_and_limit(ho):
    rng = np.random.default_rng(2)
    amin, amax = [-1, -1, -1], [1, 1, 1]
    for _ in range(500):
        d = rng.normal(size=3)
        d /= np.linalg.norm(d)
        r = float(np.exp(rng.uniform(math.log(1e-3), math.log(1e6))))
        x = ho.contract(d * r, amin, amax).astype(np.float64)
        assert (x >= 0).all() and (x <= 1).all()                 # paper: range (0,1), PAPER.md:70 (pins reading A1)
        rad = np.linalg.norm(x - 0.5)
        expect = 0.25 * r if r <= 1 else 0.25 * (2 - 1 / r)      # Mip-NeRF360 contraction scaled by 0.25
        assert abs(rad - expect) < 1e-6
        assert np.allclose((x - 0.5) / rad, d, atol=1e-4)        # direction preserved
    # continuity at |p'| = 1 and limit |x - 0.5| -> 0.5
    a = ho.contract([np.nextafter(np.float32(1), np.float32(0)), 0, 0], amin, amax)
    b = ho.contract([np.nextafter(np.float32(1), np.float32(2)), 0, 0], amin, amax)
    assert abs(float(a[0]) - float(b[0])) < 1e-6 and abs(float(a[0]) - 0.75) < 1e-6
    far = ho.contract([1e8, 0, 0], amin, amax)
    assert abs(float(far[0]) - 1.0) < 1e-6


def test_contract_uses_aabb_centre_and_half_extent(ho):
    x = ho.contract([3.0, 1.0, -1.0], [1, 0, -3], [5, 2, 1])        # centre (3,1,-1) -> 0.5
    assert np.allclose(x, 0.5)
    x = ho.contract([5.0, 1.0, -1.0], [1, 0, -3], [5, 2, 1])        # +x face: p' = (1,0,0) -> 0.75
    assert np.allclose(x, [0.75, 0.5, 0.5])
