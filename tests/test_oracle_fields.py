"""Pins for the neural-field half of the oracle (DESIGN.md §2 D3-D7): grid interpolation invariants I1/I2
(north_star), hash index vs 64-bit integer arithmetic, direction encoding special values, MLP vs a textbook
numpy matmul chain, aggregation closed forms, and the paper's "w/o Neural" fallback."""
import math

import numpy as np
import pytest


def _grid(synth, res, log2_table):
    return synth.GridSpec(list(res), log2_table)


def test_grid_layout_dense_rule_and_sizes(ho, synth):
    # cfg 1 has its first 2 levels dense, 117,048 entries; cfg 2-5 first 5 dense, bg 8 levels 2.94M
    g1 = _grid(synth, synth.RES_8, 14)
    total, sizes, offs, dense = ho.grid_layout(g1)
    assert dense.tolist() == [True, True] + [False] * 6
    assert total == 4920 + 13824 + 6 * 16384 == 117048 == g1.n_entries()
    assert sizes[0] == 4920 and (sizes % 8 == 0).all()          # 17^3 = 4913 rounded up to a multiple of 8
    assert (offs == np.concatenate([[0], np.cumsum(sizes)[:-1]])).all()
    g2 = _grid(synth, synth.RES_16, 19)
    total2, sizes2, _, dense2 = ho.grid_layout(g2)
    assert dense2.sum() == 5 and (sizes2[5:] == 2 ** 19).all() and total2 == g2.n_entries()
    assert abs(total2 - 6.10e6) < 0.01e6                         # "6.10M entries"
    gb = _grid(synth, synth.RES_BG8, 19)
    assert abs(ho.grid_layout(gb)[0] - 2.94e6) < 0.01e6


def test_hash_index_against_64bit_integer_arithmetic(ho, synth):
    g = _grid(synth, [2047], 19)                                 # (2048)^3 > 2^19 -> hashed
    T = 1 << 19
    coords = [(0, 0, 0), (1, 0, 0), (0, 1, 0), (0, 0, 1), (2047, 2047, 2047), (123, 456, 789), (2048, 1, 2048),
              (1000, 2000, 3), (17, 2048, 999), (5, 5, 5), (2048, 2048, 2048)]
    seen = set()
    for vx, vy, vz in coords:
        ref = ((vx * 1) % 2 ** 32) ^ ((vy * 2654435761) % 2 ** 32) ^ ((vz * 805459861) % 2 ** 32)
        ref &= T - 1
        got = ho.grid_index(g, 0, vx, vy, vz)
        assert got == ref
        seen.add(got)
    assert len(seen) > 8                                          # not a constant
    gd = _grid(synth, [16], 19)                                   # dense: x fastest, then y, then z
    assert ho.grid_index(gd, 0, 3, 0, 0) == 3
    assert ho.grid_index(gd, 0, 0, 1, 0) == 17
    assert ho.grid_index(gd, 0, 0, 0, 1) == 17 * 17
    assert ho.grid_index(gd, 0, 16, 16, 16) == 17 ** 3 - 1


@pytest.mark.parametrize("log2_table", [19, 9])                   # all-dense, and level 1+ hashed
def test_I1_exact_value_at_vertices(ho, synth, log2_table):
    res = [4, 8, 16]
    g = _grid(synth, res, log2_table)
    total, sizes, offs, dense = ho.grid_layout(g)
    assert dense[0] and (log2_table == 19) == bool(dense[2])
    rng = np.random.default_rng(3)
    table = rng.uniform(-1, 1, size=(total, 2)).astype(np.float32)
    for _ in range(60):
        # x = v / N is exact for power-of-two N; every level sees a vertex exactly when v is on the coarsest grid
        v = rng.integers(0, 5, size=3)
        x = v.astype(np.float32) / np.float32(4)
        feat = ho.grid_encode(g, table, x)
        for l, N in enumerate(res):
            vv = v * (N // 4)
            e = ho.grid_index(g, l, int(vv[0]), int(vv[1]), int(vv[2]))
            assert (feat[2 * l:2 * l + 2] == table[offs[l] + e]).all()       # bit-exact (weights are 0/1)


def test_I2_affine_table_gives_affine_output_dense(ho, synth):
    res = [5, 9, 14]
    g = _grid(synth, res, 20)                                    # all dense
    total, sizes, offs, dense = ho.grid_layout(g)
    assert dense.all()
    a = np.array([0.3, -0.7, 1.1]); b = 0.25
    table = np.zeros((total, 2), np.float32)
    for l, N in enumerate(res):
        n1 = N + 1
        vz, vy, vx = np.meshgrid(np.arange(n1), np.arange(n1), np.arange(n1), indexing="ij")
        val = (a[0] * vx + a[1] * vy + a[2] * vz) / N + b        # f(v/N), f affine
        idx = (vx + n1 * (vy + n1 * vz)).ravel()
        table[offs[l] + idx, 0] = val.ravel()
        table[offs[l] + idx, 1] = 1.0                            # constant table -> weights sum to 1
    rng = np.random.default_rng(4)
    for _ in range(200):
        x = rng.uniform(0, 1, 3).astype(np.float32)
        feat = ho.grid_encode(g, table, x).reshape(-1, 2)
        assert np.allclose(feat[:, 0], a @ x.astype(np.float64) + b, atol=3e-6)
        assert np.allclose(feat[:, 1], 1.0, atol=3e-7)
    # boundary x = 1: cell index clamps to N-1 with w = 1 -> still the vertex value
    feat = ho.grid_encode(g, table, np.ones(3, np.float32)).reshape(-1, 2)
    assert np.allclose(feat[:, 0], a.sum() + b, atol=3e-6)


def test_trilinear_against_numpy_reference_on_hashed_level(ho, synth):
    g = _grid(synth, [37], 10)
    total, _, offs, dense = ho.grid_layout(g)
    assert not dense[0]
    rng = np.random.default_rng(5)
    table = rng.uniform(-1, 1, size=(total, 2)).astype(np.float32)
    for _ in range(100):
        x = rng.uniform(0, 1, 3).astype(np.float32)
        u = x.astype(np.float64) * 37
        i = np.minimum(np.floor(u), 36).astype(int)
        w = u - i
        ref = np.zeros(2)
        for k in range(8):
            b = np.array([k & 1, (k >> 1) & 1, (k >> 2) & 1])
            wt = np.prod(np.where(b == 1, w, 1 - w))
            e = ho.grid_index(g, 0, *(int(q) for q in (i + b)))
            ref += wt * table[e].astype(np.float64)
        assert np.allclose(ho.grid_encode(g, table, x), ref, atol=2e-6)


def test_fp16_table_features_are_halves(ho, synth):
    g = _grid(synth, [4, 8, 16, 32], 9)
    total = ho.grid_layout(g)[0]
    rng = np.random.default_rng(6)
    t32 = rng.uniform(-1, 1, size=(total, 2)).astype(np.float32)
    t16 = t32.astype(np.float16)
    x = rng.uniform(0, 1, 3).astype(np.float32)
    f16 = ho.grid_encode(g, t16, x, fp16=True)
    f32 = ho.grid_encode(g, t16.astype(np.float32), x, fp16=False)
    assert (f16 == f32.astype(np.float16).astype(np.float32)).all()     # = fp32 result rounded once to half


def test_dir_pe_special_directions_and_layout(ho):
    pe = ho.dir_pe([1, 0, 0])
    # k = 0: sin(pi d) = (0,0,0), cos(pi d) = (-1, 1, 1); k >= 1: sin = 0, cos(2^k pi) = 1
    assert np.allclose(pe[0:3], 0, atol=1e-7) and np.allclose(pe[3:6], [-1, 1, 1], atol=1e-7)
    for k in range(1, 4):
        assert np.allclose(pe[6 * k:6 * k + 3], 0, atol=1e-6) and np.allclose(pe[6 * k + 3:6 * k + 6], 1, atol=1e-7)
    pe = ho.dir_pe([0, 0.5, -0.25])
    assert np.allclose(pe[0:3], [0, 1, -math.sqrt(0.5)], atol=1e-7)      # sin(pi d)
    assert np.allclose(pe[3:6], [1, 0, math.sqrt(0.5)], atol=1e-7)       # cos(pi d)
    assert np.allclose(pe[6:9], [0, 0, -1], atol=1e-7)                   # sin(2 pi d)
    rng = np.random.default_rng(7)
    d = rng.normal(size=3); d /= np.linalg.norm(d)
    pe = ho.dir_pe(d.astype(np.float32)).reshape(4, 2, 3)
    assert np.allclose(pe[:, 0] ** 2 + pe[:, 1] ** 2, 1, atol=1e-6)
    d32 = d.astype(np.float32).astype(np.float64)
    for k in range(4):
        assert np.allclose(pe[k, 0], np.sin(np.pi * 2 ** k * d32), atol=1e-6)
        assert np.allclose(pe[k, 1], np.cos(np.pi * 2 ** k * d32), atol=1e-6)


def test_view_dir_is_unit_and_points_from_camera(ho):
    d = ho.view_dir([1, 2, 3], [1, 2, -1])
    assert np.allclose(d, [0, 0, 1])
    d = ho.view_dir([0.3, -1.2, 2.0], [4, 0, 0])
    ref = np.array([0.3 - 4, -1.2, 2.0]); ref /= np.linalg.norm(ref)
    assert np.allclose(d, ref, atol=1e-7) and abs(np.linalg.norm(d) - 1) < 1e-6


@pytest.mark.parametrize("spec", [(16, 32, 1, 8), (56, 64, 2, 3), (40, 64, 1, 3), (7, 5, 3, 2)])
def test_mlp_matches_numpy_matmul_chain(ho, synth, spec):
    m = synth.MlpSpec(*spec)
    rng = np.random.default_rng(8)
    w = rng.normal(0, 0.3, m.n_weights()).astype(np.float32)
    x = rng.normal(0, 1, m.in_dim).astype(np.float32)
    h = x.astype(np.float64)
    off = 0
    shapes = m.layer_shapes()
    for li, (o, i) in enumerate(shapes):
        W = w[off:off + o * i].reshape(o, i).astype(np.float64); off += o * i
        h = W @ h
        if li < len(shapes) - 1:
            h = np.maximum(h, 0)
    got = ho.mlp_forward(m, w, x)
    assert np.allclose(got, h, atol=1e-5, rtol=1e-5)
    # no bias: zero input -> zero output exactly
    assert (ho.mlp_forward(m, w, np.zeros(m.in_dim, np.float32)) == 0).all()


def test_mlp_fp16_path_matches_explicit_half_casts(ho, synth):
    m = synth.MlpSpec(32, 64, 2, 8)
    rng = np.random.default_rng(9)
    w = rng.normal(0, 0.2, m.n_weights()).astype(np.float16)
    x = rng.normal(0, 0.5, m.in_dim).astype(np.float16).astype(np.float32)
    h = x.astype(np.float64)
    off = 0
    shapes = m.layer_shapes()
    for li, (o, i) in enumerate(shapes):
        W = w[off:off + o * i].reshape(o, i).astype(np.float64); off += o * i
        h = W @ h
        if li < len(shapes) - 1:
            h = np.maximum(h, 0).astype(np.float16).astype(np.float64)      # hidden rounded to half after ReLU
    got = ho.mlp_forward(m, w, x, fp16=True)
    assert np.allclose(got, h, atol=2e-3, rtol=2e-3)     # a half-ulp flip of a hidden unit is allowed, no more


def test_aggregate_closed_forms(ho):
    raw = np.array([0.3, 0.1, -0.2, 0.05, 2.0, 0.0, 0.0, 0.0, -1.0, 0.5, 2.0], np.float32)
    at = ho.aggregate(raw, s_e=-4.0, a_e=0.7, c_e=[0.2, -0.3, 0.1])
    sg = lambda v: 1 / (1 + math.exp(-v))
    assert np.allclose(at[0:3], [sg(0.1 - 4), sg(-0.2 - 4), sg(0.05 - 4)], atol=1e-7)   # s = sigma(s_n + s_e)
    assert np.allclose(at[3:7], [1, 0, 0, 0])                                           # r = r_n/|r_n|
    assert abs(at[7] - sg(1.0)) < 1e-7                                                  # alpha
    assert np.allclose(at[8:11], [sg(-0.8), sg(0.2), sg(2.1)], atol=1e-7)               # c
    # alpha_n = 0 -> sigma(alpha_e); quaternion normalised in (w,x,y,z) order
    raw2 = np.zeros(11, np.float32); raw2[4:8] = [1, 2, 3, 4]
    at2 = ho.aggregate(raw2, 0.0, 1.3, [0, 0, 0])
    assert abs(at2[7] - sg(1.3)) < 1e-7
    assert np.allclose(at2[3:7], np.array([1, 2, 3, 4]) / math.sqrt(30), atol=1e-7)
    # zero quaternion: denominator max(|r|, 1e-12) -> r = 0, no NaN
    at3 = ho.aggregate(np.zeros(11, np.float32), 0.0, 0.0, [0, 0, 0])
    assert (at3[3:7] == 0).all() and np.isfinite(at3).all()


def test_zero_tables_fall_back_to_isotropic_diffuse(ho, synth):
    # without the neural components the model is isotropic Gaussians with diffuse shading.
    # Geometry: zero geo table + no bias -> raw geometry exactly 0 -> s = sigma(s_e) on all three axes.
    s = synth.tiny_scene(n=40)
    s.geo_table = np.zeros_like(s.geo_table)
    s.app_table = np.zeros_like(s.app_table)
    s.app_w = np.zeros_like(s.app_w)                  # kills the view-dependent PE part too
    osc = ho.OracleScene(s)
    cam = s.cameras[0]
    mask, idx = ho.stage_cull(osc, cam, cam.W, cam.H)
    raw = ho.stage_query(osc, cam, idx)
    assert (raw == 0).all()
    attrs = ho.stage_aggregate(osc, idx, raw)
    sg = lambda v: 1 / (1 + np.exp(-v.astype(np.float64)))
    assert np.allclose(attrs[:, 0], sg(s.scale_logit[idx]), atol=1e-7)
    assert (attrs[:, 0] == attrs[:, 1]).all() and (attrs[:, 1] == attrs[:, 2]).all()      # isotropic
    assert np.allclose(attrs[:, 7], sg(s.opacity_logit[idx]), atol=1e-7)
    assert np.allclose(attrs[:, 8:11], sg(s.rgb_logit[:, idx].T), atol=1e-7)              # diffuse colour
    # zero quaternion projects like the identity rotation: Sigma = s^2 I (checked in test_oracle_raster)


def test_query_point_equals_its_parts(ho, synth):
    # wiring pin: f_geo -> Phi_geo, f_rad (+) PE -> Phi_c (reading A7), outputs in (alpha, s3, r4, c3) order
    s = synth.tiny_scene(n=8, table_amp=1.0)
    osc = ho.OracleScene(s)
    cam = s.cameras[1]
    o = ho.camera_center(cam)
    p = s.pos[:, 3]
    x = ho.contract(p, s.aabb_min, s.aabb_max)
    fg = ho.grid_encode(s.geo_grid, s.geo_table, x)
    fa = ho.grid_encode(s.app_grid, s.app_table, x)
    pe = ho.dir_pe(ho.view_dir(p, o))
    geo = ho.mlp_forward(s.geo_mlp, s.geo_w, fg)
    app = ho.mlp_forward(s.app_mlp, s.app_w, np.concatenate([fa, pe]))
    raw = ho.query_point(osc, p, o)
    assert (raw[:8] == geo).all() and (raw[8:] == app).all()
    assert np.abs(raw).max() > 1e-3
