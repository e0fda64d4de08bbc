"""Pins for the oracle's ablation switches (PAPER.md:214-223 Table 5, :233-237, :259): each switch must equal the
full pass run on a scene that realises the ablation by construction — not by the switch."""
import copy

import numpy as np


def _scene(synth):
    return synth.make_scene(3, n_gaussians=4000, width=96, height=64, n_cameras=1, table_amp=0.5)


def test_no_neural_equals_zero_tables(ho, synth):
    # without the neural part the Gaussians are the explicit ones. No biases anywhere, so zero
    # tables give zero decoder outputs... except the appearance decoder, which also sees the direction encoding:
    # zero its weights too.
    s = _scene(synth)
    z = copy.copy(s)
    z.geo_table = np.zeros_like(s.geo_table)
    z.app_table = np.zeros_like(s.app_table)
    z.app_w = np.zeros_like(s.app_w)
    a = ho.render(ho.OracleScene(s), s.cameras[0], ablation=ho.ABL_NO_NEURAL)
    b = ho.render(ho.OracleScene(z), s.cameras[0])
    assert (a["raw"] == 0).all() and (b["raw"] == 0).all()
    assert (a["out"] == b["out"]).all() and (a["list_id"] == b["list_id"]).all()
    # isotropic, identity rotation
    assert (a["attrs"][:, 0] == a["attrs"][:, 1]).all() and (a["attrs"][:, 1] == a["attrs"][:, 2]).all()


def test_no_explicit_equals_zero_logits(ho, synth):
    s = _scene(synth)
    z = copy.copy(s)
    z.rgb_logit = np.zeros_like(s.rgb_logit)
    z.scale_logit = np.zeros_like(s.scale_logit)
    z.opacity_logit = np.zeros_like(s.opacity_logit)
    s2 = synth.make_scene(3, n_gaussians=4000, width=24, height=16, n_cameras=1, table_amp=0.5)   # sigma(0)=0.5 splats are huge
    z2 = copy.copy(s2)
    z2.rgb_logit, z2.scale_logit, z2.opacity_logit = (np.zeros_like(s2.rgb_logit), np.zeros_like(s2.scale_logit),
                                                      np.zeros_like(s2.opacity_logit))
    a = ho.render(ho.OracleScene(s2), s2.cameras[0], ablation=ho.ABL_NO_EXPLICIT)
    b = ho.render(ho.OracleScene(z2), s2.cameras[0])
    assert (a["attrs"] == b["attrs"]).all() and (a["out"] == b["out"]).all()
    assert z.n == s.n


def test_no_cull_moves_work_not_pixels(ho, synth):
    s = _scene(synth)
    osc = ho.OracleScene(s)
    full = ho.render(osc, s.cameras[0])
    nc = ho.render(osc, s.cameras[0], ablation=ho.ABL_NO_CULL)
    assert len(nc["vis_idx"]) == s.n > len(full["vis_idx"])          # every stored Gaussian was queried
    assert (nc["out"] == full["out"]).all() and (nc["T"] == full["T"]).all()
    assert nc["D"] == full["D"] and (nc["list_id"] == full["list_id"]).all() and (nc["ranges"] == full["ranges"]).all()
    # queried values of the Gaussians the full pass also saw are the same numbers
    assert (nc["raw"][full["vis_idx"]] == full["raw"]).all()


def test_no_background_is_foreground_only(ho, synth):
    s = _scene(synth)
    osc = ho.OracleScene(s)
    full = ho.render(osc, s.cameras[0])
    nb = ho.render(osc, s.cameras[0], ablation=ho.ABL_NO_BG)
    assert (nb["out"] == full["cfg"]).all() and not nb["bg_mask"].any()
    assert full["bg_mask"].any() and (full["out"] != full["cfg"]).any()
