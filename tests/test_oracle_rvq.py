"""Pins for the decode of the compressed explicit Gaussians (PAPER.md:227-229 items 1-2; DESIGN.md §2 D1'):
positions from IEEE binary16, properties as the stage-ordered binary32 sum of one codebook row per R-VQ stage.
None of the expected values below comes from the oracle (hand-written numbers, numpy's own float16, exact rational
arithmetic)."""
from fractions import Fraction
from types import SimpleNamespace as NS

import numpy as np
import pytest


def _rvq(pos_h, codes, books):
    return NS(pos_h=np.asarray(pos_h, np.uint16), codes=np.asarray(codes, np.uint16),
              codebooks=np.asarray(books, np.float32))


def test_half_positions_hand_values(ho):
    # binary16 patterns whose values are known by hand: 1, -2, smallest subnormal 2^-24, largest finite 65504,
    # 1/3 rounded to 11 bits (0x3555 = 1365/4096), -0, 0.1 rounded (0x2E66 = 1638/16384)
    bits = [0x3C00, 0xC000, 0x0001, 0x7BFF, 0x3555, 0x8000, 0x2E66, 0x0400, 0x03FF]
    want = [1.0, -2.0, 2.0 ** -24, 65504.0, 1365.0 / 4096.0, -0.0, 1638.0 / 16384.0, 2.0 ** -14, 1023.0 * 2.0 ** -24]
    n = len(bits)
    pos_h = np.array([bits, bits[::-1], bits], np.uint16)
    d = ho.decode_explicit(_rvq(pos_h, np.zeros((1, n)), np.zeros((1, 1, 5))))
    assert (d["pos"][0] == np.array(want, np.float32)).all()
    assert (d["pos"][1] == np.array(want[::-1], np.float32)).all()      # axis a reads row a: SoA [3][N]
    assert np.signbit(d["pos"][0][5])


def test_half_positions_every_finite_pattern_matches_numpy_float16(ho):
    bits = np.arange(65536, dtype=np.uint16)
    finite = (bits & 0x7C00) != 0x7C00
    bits = bits[finite]
    n = len(bits)
    d = ho.decode_explicit(_rvq(np.stack([bits, bits, bits]), np.zeros((1, n)), np.zeros((1, 1, 5))))
    want = bits.view(np.float16).astype(np.float32)                       # numpy's converter, not the oracle's
    assert (d["pos"][2].view(np.uint32) == want.view(np.uint32)).all()


def test_single_stage_is_a_row_lookup_and_columns_map_to_attributes(ho):
    # one stage: x = C_0[k]. Column d of row k holds 10 k + d, so a wrong row, column or output array shows
    K, n = 7, 23
    books = (10.0 * np.arange(K)[:, None] + np.arange(5)[None, :]).astype(np.float32)[None]
    codes = (np.arange(n) * 3 % K)[None]
    d = ho.decode_explicit(_rvq(np.zeros((3, n)), codes, books))
    k = codes[0]
    assert (d["scale_logit"] == 10.0 * k + 0).all()
    assert (d["opacity_logit"] == 10.0 * k + 1).all()
    for c in range(3):
        assert (d["rgb_logit"][c] == 10.0 * k + 2 + c).all()
    assert (d["pos"] == 0).all()


def test_codes_are_stage_major(ho):
    # codes[s][i]: stage 0 contributes k, stage 1 contributes 100 k'; a transposed read mixes them up
    K, n = 5, 10
    books = np.zeros((2, K, 5), np.float32)
    books[0] = np.arange(K)[:, None]
    books[1] = 100.0 * np.arange(K)[:, None]
    c0 = np.arange(n) % K
    c1 = (np.arange(n) * 2 + 1) % K
    d = ho.decode_explicit(_rvq(np.zeros((3, n)), np.stack([c0, c1]), books))
    assert (d["scale_logit"] == c0 + 100.0 * c1).all()
    assert (d["rgb_logit"][2] == c0 + 100.0 * c1).all()


def test_sum_is_binary32_left_to_right_in_stage_order(ho):
    # (1e8 + -1e8) + 1 = 1 in binary32, while 1e8 + (-1e8 + 1) = 0 (1e8's ulp is 8) and any order that adds the 1 to
    # +-1e8 first loses it; 2^24 + 1 + 1: left to right stays 2^24 (each +1 is a tie to even), exact sum is 2^24 + 2
    books = np.zeros((3, 2, 5), np.float32)
    books[0, 0], books[1, 0], books[2, 0] = 1e8, -1e8, 1.0
    books[0, 1], books[1, 1], books[2, 1] = 2.0 ** 24, 1.0, 1.0
    codes = np.array([[0, 1], [0, 1], [0, 1]])
    d = ho.decode_explicit(_rvq(np.zeros((3, 2)), codes, books))
    assert d["scale_logit"][0] == 1.0 and d["opacity_logit"][0] == 1.0
    assert d["scale_logit"][1] == 2.0 ** 24 and d["rgb_logit"][1][1] == 2.0 ** 24


def test_two_stage_sum_is_the_correctly_rounded_exact_sum(ho):
    # one binary32 addition is the exact rational sum rounded to nearest even: check against Fractions
    rng = np.random.default_rng(11)
    K, n = 16, 64
    books = (rng.normal(0, 1, (2, K, 5)) * np.array([1.0, 2.0 ** -9])[:, None, None]).astype(np.float32)
    codes = rng.integers(0, K, (2, n))
    d = ho.decode_explicit(_rvq(np.zeros((3, n)), codes, books))
    got = np.stack([d["scale_logit"], d["opacity_logit"], *d["rgb_logit"]], axis=1)
    for i in range(n):
        for c in range(5):
            exact = Fraction(float(books[0, codes[0, i], c])) + Fraction(float(books[1, codes[1, i], c]))
            g = Fraction(float(got[i, c]))
            lo, hi = np.nextafter(got[i, c], np.float32(-np.inf)), np.nextafter(got[i, c], np.float32(np.inf))
            assert abs(g - exact) <= abs(Fraction(float(lo)) - exact) and abs(g - exact) <= abs(Fraction(float(hi)) - exact)


def test_out_of_range_code_is_rejected(ho):
    with pytest.raises(ValueError):
        ho.decode_explicit(_rvq(np.zeros((3, 4)), [[0, 1, 2, 3]], np.zeros((1, 3, 5))))


def test_encoder_round_trip_and_residual_refinement(ho, synth):
    # rows drawn from a product of per-stage alphabets are reproduced exactly by a codebook holding those alphabets;
    # and on generic rows every extra stage of the synthetic encoder lowers the reconstruction error
    s = synth.make_scene(1, n_gaussians=2048, n_cameras=1)
    errs = []
    for stages in (1, 2, 4, 6):
        c = synth.compress_explicit(s, stages=stages, codebook_size=32, seed=3)
        d = ho.decode_explicit(c.explicit_rvq)
        rows = np.stack([d["scale_logit"] - s.scale_logit, d["opacity_logit"] - s.opacity_logit,
                         *(d["rgb_logit"] - s.rgb_logit)])
        errs.append(float(np.sqrt((rows.astype(np.float64) ** 2).mean())))
        assert (d["pos"] == np.asarray(s.pos).astype(np.float16).astype(np.float32)).all()
        assert np.abs(d["pos"] - s.pos).max() <= 2.0 ** -11 * np.abs(s.pos).max()     # half an ulp of binary16
    assert errs[0] > errs[1] > errs[2] > errs[3]


def test_render_of_compressed_scene_is_render_of_decoded_arrays(ho, synth):
    # the compressed scene differs from a plain scene only in where the explicit arrays come from
    s = synth.compress_explicit(synth.tiny_scene(n=40, W=24, H=24), stages=3, codebook_size=8)
    d = ho.decode_explicit(s.explicit_rvq)
    import copy
    plain = copy.copy(s)
    plain.explicit_rvq = None
    plain.pos, plain.scale_logit, plain.opacity_logit, plain.rgb_logit = (d["pos"], d["scale_logit"],
                                                                          d["opacity_logit"], d["rgb_logit"])
    a = ho.render(ho.OracleScene(s), s.cameras[0])
    b = ho.render(ho.OracleScene(plain), s.cameras[0])
    assert (a["out"] == b["out"]).all() and (a["list_id"] == b["list_id"]).all()
    src = ho.render(ho.OracleScene(synth.tiny_scene(n=40, W=24, H=24)), s.cameras[0])
    assert not (a["out"] == src["out"]).all()             # the codes are what is rendered, not the source arrays
