"""Pins for the 8-bit min-max table decode of the compressed model (PAPER.md:227-229 item 3; DESIGN.md §2 D3').
The decode is value = fma(code, step, min) per level and feature; everything after it is the fp16 path."""
import numpy as np


def _half(v):
    return np.asarray(v, np.float32).astype(np.float16).astype(np.float32)


def test_decode_equals_fp32_table_of_decoded_values(ho, synth):
    # the 8-bit path must be the fp32 path run on the table of decoded values, then rounded to fp16: same blend,
    # same order, only the storage differs. The fp32 route is pinned by test_oracle_fields.py (I1, I2).
    rng = np.random.default_rng(5)
    grid = synth.GridSpec([4, 7, 12, 21, 37, 64], 10)          # 3 dense + 3 hashed levels
    n = grid.n_entries()
    codes = rng.integers(0, 256, size=(n, 2), dtype=np.uint8)
    q = np.zeros((grid.levels, 2, 2), np.float32)
    q[..., 0] = rng.uniform(-1, 0, size=(grid.levels, 2))
    q[..., 1] = rng.uniform(1e-3, 8e-3, size=(grid.levels, 2))
    decoded = np.zeros((n, 2), np.float32)
    off = 0
    for l, sz in enumerate(grid.level_sizes()):
        for f in range(2):   # fma in exact arithmetic: code * step is exact in float64, one rounding to float32
            decoded[off:off + sz, f] = (codes[off:off + sz, f].astype(np.float64) * np.float64(q[l, f, 1]) +
                                        np.float64(q[l, f, 0])).astype(np.float32)
        off += sz
    for _ in range(200):
        x = rng.uniform(0, 1, 3).astype(np.float32)
        a = ho.grid_encode(grid, codes, x, q=q)
        b = _half(ho.grid_encode(grid, decoded, x, fp16=False))
        assert (a == b).all()


def test_codes_reproduce_min_and_max_at_vertices(ho, synth):
    grid = synth.GridSpec([4, 8], 12)                           # both dense
    n = grid.n_entries()
    q = np.array([[[-0.25, 0.002], [0.5, 0.001]], [[-1.0, 0.004], [0.0, 0.003]]], np.float32)
    for code in (0, 255, 37):
        codes = np.full((n, 2), code, np.uint8)
        x = np.array([0.5, 0.25, 0.75], np.float32)             # a vertex of both levels
        got = ho.grid_encode(grid, codes, x, q=q)
        want = _half((np.float64(code) * q[..., 1].astype(np.float64) + q[..., 0].astype(np.float64)).astype(np.float32))
        assert (got.reshape(2, 2) == want).all()                # constant table -> the decoded constant, exactly


def test_quantised_scene_is_close_to_its_source(ho, synth):
    # min-max quantisation error is at most step / 2 per entry: the render of the quantised scene must stay within
    # the corresponding bound of the fp16 scene it was made from (and must not be identical: the codes are used)
    s = synth.make_scene(3, n_gaussians=3000, width=96, height=64, n_cameras=1, table_amp=0.5)
    sq = synth.quantize8(s)
    assert sq.geo_table.dtype == np.uint8 and sq.geo_q.shape == (16, 2, 2)
    a = ho.render(ho.OracleScene(s), s.cameras[0])
    b = ho.render(ho.OracleScene(sq), sq.cameras[0])
    d = np.abs(a["raw"] - b["raw"]).max()
    assert 0.0 < d < 1e-2
    assert (a["mask"] == b["mask"]).all()                       # culling does not depend on the fields
