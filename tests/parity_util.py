"""Element-by-element comparison of one GPU frame (C-ABI debug exports) with the oracle's frame.

Three protocols, all against the same oracle:

* `compare_frame(..., exact_geometry=True)` — the exact path (HYRF_MLP_FMA: decoders in the oracle's fma order):
  masks, geometry logits, records, rectangles, D, tile ranges and per-tile lists BIT-EXACT; image within
  BASELINE.json's tolerance (2e-3 max-abs / 1e-4 mean-abs per channel in fp32, 1e-2 max-abs with fp16 parameters).
* `compare_handoff(...)` — the tensor-core paths: stages 1-3 against the oracle by tolerance
  (mask bit-exact, raw logits within 2e-3), then the oracle's stages O7-O10 are run ON THE GPU'S OWN stage-3
  attributes and must reproduce the GPU's records, rectangles, D, tile ranges and per-tile lists BIT FOR BIT and its
  image at the exact path's tolerance. Given the attributes, nothing after stage 3 is allowed to differ.
* the end-to-end part of `compare_handoff` — what the 2e-3 of logit noise does to the picture. The pass is
  discontinuous (alpha < 1/255 skip, T' < 1e-4 stop, tau_T test, 3-sigma rectangle), so the comparison is split by
  CAUSE, decided exactly instead of by widened margins: a pixel whose discrete decisions are the same in the oracle's
  two renders (its own attributes / the GPU's attributes: same evaluated and blended pair counts, same background
  decision) is a smooth function of the attributes and must be within the tolerance; the other pixels ("flipped")
  are counted, reported and bounded by the worst case of their cause.

Fragile pixels, exact comparisons only: the rasterizer's exp is the MUFU ex2.approx (2 ulp) against
the oracle's D6 soft exponential, so a pair within 5e-8 of the alpha = 1/255 skip, a stop decision within 5e-5
relative of T' = 1e-4 or a final T within 1e-5 of tau_T may be decided differently. Per cause: an alpha flip moves a
channel by at most alpha T_k |c_k - C_behind| <= 1/255; a stop flip by at most alpha T c <= 0.99e-2 (T' < 1e-4 with
alpha <= 0.99 means T <= 1e-2); a tau_T flip by up to T c_s and is excluded. The expected fragile fraction is
n_eval * 2 m / (alpha_thr * L) with m = 5e-8, alpha_thr = 1/255, L ~ 5 the spread of ln(alpha) over the evaluated
pairs: 5e-6 per evaluated pair, i.e. 0.09 % at 170 evaluated pairs per pixel (config 3) — the bound below is three
times that estimate for the frame at hand (never below 0.1 %), not a constant tuned to a measurement.
"""
import json
import os

import numpy as np

ALPHA_THR = 1.0 / 255.0
M_ALPHA, M_STOP, M_TAU = 5e-8, 5e-5, 1e-5     # fragility margins of the exact comparisons
ALPHA_FLIP, STOP_FLIP = 1.0 / 255.0, 1e-2     # worst-case change of a channel per flipped decision (derivation above)

_STATS = []


def record_stats(label, st):
    """Append one frame's parity statistics to gpurun_out/parity_stats.jsonl (read back into BASELINE.md §3)."""
    _STATS.append((label, st))
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    try:
        os.makedirs(os.path.join(root, "gpurun_out"), exist_ok=True)
        with open(os.path.join(root, "gpurun_out", "parity_stats.jsonl"), "a") as f:
            f.write(json.dumps({"label": label, **{k: v for k, v in st.items() if not isinstance(v, np.ndarray)}}) + "\n")
    except OSError:
        pass


def bits_equal(a, b):
    a = np.ascontiguousarray(a, np.float32).view(np.uint32)
    b = np.ascontiguousarray(b, np.float32).view(np.uint32)
    return a == b


def fragile_bound(orc):
    """Three times the expected fraction of pixels holding a pair inside the alpha margin (module docstring)."""
    n_eval = float(orc["n_eval"].mean()) if "n_eval" in orc else 0.0
    return max(1e-3, 3.0 * n_eval * 2.0 * M_ALPHA / (ALPHA_THR * 5.0))


def _check_stage123(orc, gpu, exact, fp16, label, st):
    assert (gpu["mask"] == orc["mask"]).all(), f"{label}: visibility mask differs"
    assert (gpu["vis_idx"] == orc["vis_idx"]).all(), f"{label}: visible index list differs"
    V = len(orc["vis_idx"])
    st["V"] = V
    assert int(gpu["counters"][1]) == V
    if not V:
        return
    raw_g, raw_o, at_g, at_o = gpu["raw"], orc["raw"], gpu["attrs"], orc["attrs"]
    st["raw_geo_maxdiff"] = float(np.abs(raw_g[:, :8] - raw_o[:, :8]).max())
    st["raw_app_maxdiff"] = float(np.abs(raw_g[:, 8:] - raw_o[:, 8:]).max())
    st["attrs_maxdiff"] = float(np.abs(at_g - at_o).max())
    if exact:
        assert bits_equal(raw_g[:, :8], raw_o[:, :8]).all(), f"{label}: geometry decoder outputs not bit-exact"
        assert bits_equal(at_g[:, :8], at_o[:, :8]).all(), f"{label}: scale/rotation/opacity not bit-exact"
        app_tol = 2e-3 if fp16 else 2e-5       # sinpi/cospi routines differ by ulps; fp16 can flip a half rounding
        assert st["raw_app_maxdiff"] <= app_tol, f"{label}: appearance logits differ by {st['raw_app_maxdiff']}"
        assert np.abs(at_g[:, 8:] - at_o[:, 8:]).max() <= app_tol
    else:
        assert st["raw_geo_maxdiff"] <= 2e-3 and st["raw_app_maxdiff"] <= 2e-3, f"{label}: raw logits {st}"
        # sigmoid' <= 1/4 and the unit quaternion of logits O(0.01-1): attributes follow the logits
        assert np.abs(at_g[:, [0, 1, 2, 7, 8, 9, 10]] - at_o[:, [0, 1, 2, 7, 8, 9, 10]]).max() <= 1e-3, f"{label}: attributes {st}"


def _check_lists_exact(orc, gpu, label, st, proj_cols):
    """Records, rectangles, D, ranges and per-tile lists bit for bit."""
    assert bits_equal(gpu["proj"][:, :proj_cols], orc["proj"][:, :proj_cols]).all(), f"{label}: projected records not bit-exact"
    tiles_o = orc["tiles"]
    rg = gpu["rect"].astype(np.int64)
    tiles_g = (rg[:, 1] - rg[:, 0]) * (rg[:, 3] - rg[:, 2])
    tiles_g = np.where((rg[:, 1] > rg[:, 0]) & (rg[:, 3] > rg[:, 2]), tiles_g, 0)
    assert (tiles_g == tiles_o).all(), f"{label}: tiles touched differ"
    nz = tiles_o > 0
    assert (gpu["rect"][nz] == orc["rect"][nz]).all(), f"{label}: tile rectangles differ"
    assert int(gpu["counters"][2]) == orc["D"], f"{label}: D {int(gpu['counters'][2])} vs {orc['D']}"
    assert (gpu["ranges"] == orc["ranges"]).all(), f"{label}: tile ranges differ"
    assert (gpu["list_id"] == orc["list_id"]).all(), f"{label}: per-tile Gaussian lists differ"
    st["D"] = orc["D"]


def _check_image_exact(orc, gpu, out_gpu, tau_T, fp16, label, st, key=""):
    """GPU image against an oracle render of the SAME records: only the exp of stage 5 (and the routines of the
    background decoder) differ; fragile pixels per cause."""
    Tg, To = gpu["T"], orc["T"]
    frag_alpha = orc["m_alpha"] < M_ALPHA
    frag_stop = orc["m_stop"] < M_STOP
    frag_tau = (np.abs(To - np.float32(tau_T)) < M_TAU) & (orc["n_blend"] > 0)   # T = 1 exactly when nothing blended
    fragile = frag_alpha | frag_stop | frag_tau
    st[key + "fragile_frac"] = float(fragile.mean())
    st[key + "fragile_bound"] = fragile_bound(orc)
    tol_max = 1e-2 if fp16 else 2e-3
    diff = np.abs(out_gpu.astype(np.float64) - orc["out"].astype(np.float64))
    ok = ~fragile
    st[key + "img_max_nonfragile"] = float(diff[ok].max()) if ok.any() else 0.0
    st[key + "img_mean"] = [float(diff[..., c][ok].mean()) if ok.any() else 0.0 for c in range(3)]
    st[key + "T_max_nonfragile"] = float(np.abs(Tg - To)[ok].max()) if ok.any() else 0.0
    st[key + "n_above_1e-2"] = int((diff.max(axis=-1) > 1e-2).sum())
    assert st[key + "fragile_frac"] <= st[key + "fragile_bound"], f"{label}: too many fragile pixels {st}"
    assert st[key + "img_max_nonfragile"] <= tol_max, f"{label}: image max-abs {st}"
    assert max(st[key + "img_mean"]) <= 1e-4, f"{label}: image mean-abs {st}"
    assert st[key + "T_max_nonfragile"] <= tol_max
    # per cause: alpha flips move a channel by <= 1/255 each, a stop flip by <= 1e-2 (module docstring)
    only_alpha = frag_alpha & ~frag_stop & ~frag_tau
    with_stop = frag_stop & ~frag_tau
    st[key + "img_max_fragile"] = float(diff[fragile & ~frag_tau].max()) if (fragile & ~frag_tau).any() else 0.0
    if only_alpha.any():
        assert diff[only_alpha].max() <= tol_max + ALPHA_FLIP, f"{label}: alpha-fragile pixel off by {diff[only_alpha].max()}"
    if with_stop.any():
        assert diff[with_stop].max() <= tol_max + ALPHA_FLIP + STOP_FLIP, f"{label}: stop-fragile pixel off by {diff[with_stop].max()}"
    assert (gpu["bg_mask"].astype(bool)[ok] == orc["bg_mask"].astype(bool)[ok]).all(), f"{label}: background mask differs"


def compare_frame(orc, gpu, out_gpu, tau_T, fp16=False, exact_geometry=True, label=""):
    """Exact path. orc: dict from oracle.render; gpu: dict from HyrfScene.debug_all; out_gpu: (H, W, 3) numpy.
    (exact_geometry=False is kept for stage-level checks without per-tile lists: stages 1-3 by tolerance only.)"""
    st = {}
    _check_stage123(orc, gpu, exact_geometry, fp16, label, st)
    if exact_geometry:
        if st["V"]:
            _check_lists_exact(orc, gpu, label, st, proj_cols=7)
        else:
            st["D"] = 0
            assert int(gpu["counters"][2]) == 0
        _check_image_exact(orc, gpu, out_gpu, tau_T, fp16, label, st)
    record_stats(label, st)
    return st


def _pairs(ranges, ids):
    cnt = (ranges[:, 1].astype(np.int64) - ranges[:, 0].astype(np.int64))
    order = np.argsort(ranges[:, 0], kind="stable")
    tile = np.repeat(order, cnt[order])
    return tile * (1 << 32) + ids.astype(np.int64)


def compare_handoff(ho, osc, cam, orc, gpu, out_gpu, tau_T, fp16=True, label="", ablation=0):
    """Tensor-core paths: stages 1-3 by tolerance, stages 4-6 by hand-off (bit-exact given the GPU's attributes),
    end-to-end differences split by cause (module docstring). `orc` = oracle.render(osc, cam, ablation=ablation)."""
    st = {}
    _check_stage123(orc, gpu, False, fp16, label, st)
    # ---- hand-off: the oracle's O7-O10 on the GPU's stage-3 attributes ----
    orh = ho.render(osc, cam, attrs_override=gpu["attrs"], ablation=ablation)
    if st["V"]:
        _check_lists_exact(orh, gpu, label + " [hand-off]", st, proj_cols=10)
    _check_image_exact(orh, gpu, out_gpu, tau_T, fp16, label + " [hand-off]", st, key="handoff_")
    # ---- end to end: oracle's own attributes against the GPU's, cause by cause ----
    pg, po = _pairs(gpu["ranges"], gpu["list_id"]), _pairs(orc["ranges"], orc["list_id"])
    st["list_symdiff"] = int(len(np.setxor1d(pg, po)))
    st["list_symdiff_frac"] = st["list_symdiff"] / max(1, len(po))
    assert st["list_symdiff_frac"] < 2e-3, f"{label}: list symmetric difference {st}"
    same = (orh["n_eval"] == orc["n_eval"]) & (orh["n_blend"] == orc["n_blend"]) & (orh["bg_mask"] == orc["bg_mask"])
    flipped = ~same
    st["flipped_frac"] = float(flipped.mean())
    diff = np.abs(out_gpu.astype(np.float64) - orc["out"].astype(np.float64)).max(axis=-1)
    tol_max = 1e-2 if fp16 else 2e-3
    st["img_max_same_decisions"] = float(diff[same].max()) if same.any() else 0.0
    st["img_max_flipped"] = float(diff[flipped].max()) if flipped.any() else 0.0
    st["img_mean_all"] = float(diff.mean())
    st["n_above_1e-2"] = int((diff > 1e-2).sum())
    st["n_pixels"] = int(diff.size)
    assert st["img_max_same_decisions"] <= tol_max, f"{label}: smooth pixels differ by {st}"
    assert st["img_mean_all"] <= 1e-3, f"{label}: mean-abs {st}"
    # flipped pixels, bounded by cause: the evaluated / blended counts say how many decisions moved; every moved
    # alpha or membership decision is worth <= max(1/255, 0.011 o) < 1.2e-2 (beyond 3 sigma alpha can still
    # reach 0.011 o), a moved stop <= 1e-2; a moved tau_T decision (background mask) up to T c_s and is excluded
    bg_flip = orh["bg_mask"] != orc["bg_mask"]
    moved = (np.abs(orh["n_eval"].astype(np.int64) - orc["n_eval"].astype(np.int64)) +
             np.abs(orh["n_blend"].astype(np.int64) - orc["n_blend"].astype(np.int64)))
    chk = flipped & ~bg_flip
    if chk.any():
        bound = tol_max + 1.2e-2 * moved[chk] + STOP_FLIP
        assert (diff[chk] <= bound).all(), f"{label}: flipped pixel beyond its cause's bound {st}"
    st["bg_flipped"] = int(bg_flip.sum())
    record_stats(label, st)
    return st
