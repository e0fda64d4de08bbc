"""GPU parity tests proper: the CUDA path (through the C-ABI binding) against the CPU oracle, element by element,
on the same seeded inputs. Marked gpu: they run on the B200 box."""
import numpy as np
import pytest

from parity_util import compare_frame, compare_handoff

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2509_17083_b200 import binding
    binding.load_library()          # raises if the extension is missing: no silent fallback
    return binding


def _run(B, ho, scene, cams=None, mlp_path=None, exact=True, label="", ablation=0, raster_mode=0, bin_shift=0):
    import torch
    mlp_path = B.HYRF_MLP_FMA if mlp_path is None else mlp_path
    hs = B.HyrfScene(scene, mlp_path=mlp_path)
    hs.set_ablation(ablation)
    hs.set_raster_mode(raster_mode)
    hs.set_bin_granularity(bin_shift)
    hs.debug_enable()
    osc = ho.OracleScene(scene)
    stats = []
    for ci, cam in enumerate(cams if cams is not None else scene.cameras):
        out = hs.render(cam)
        torch.cuda.synchronize()
        gpu = hs.debug_all(cam.W, cam.H)
        orc = ho.render(osc, cam, ablation=ablation)
        lab = f"{label or scene.name} cam{ci} mlp{mlp_path} abl{ablation} r{raster_mode}"
        if exact:
            stats.append(compare_frame(orc, gpu, out.cpu().numpy(), scene.tau_T, fp16=scene.fp16, label=lab))
        else:   # tensor-core decoders: stages 1-3 by tolerance, stages 4-6 by hand-off (bit-exact lists), SURVEY H1
            stats.append(compare_handoff(ho, osc, cam, orc, gpu, out.cpu().numpy(), scene.tau_T, fp16=scene.fp16,
                                         label=lab, ablation=ablation))
    hs.close()
    return stats


def test_tiny_scene_generic_kernels_fp32(B, ho, synth):
    # run-time-shaped kernels (4 levels, hidden 16); dense + hashed levels; two cameras
    st = _run(B, ho, synth.tiny_scene(n=48, W=32, H=32))
    assert st[0]["D"] > 0


def test_tiny_scene_generic_kernels_fp16(B, ho, synth):
    _run(B, ho, synth.tiny_scene(n=64, W=48, H=40, fp16=True, seed=11))


def test_config1_full(B, ho, synth):
    st = _run(B, ho, synth.make_scene(1))
    assert st[0]["V"] == 4096


def test_config2_scaled_ragged(B, ho, synth):
    # config 2 recipe at 20k Gaussians, 200x136 (ragged right/bottom tiles), all 5 cameras
    _run(B, ho, synth.make_scene(2, n_gaussians=20_000, width=200, height=136))


def test_config2_full_two_cameras(B, ho, synth):
    s = synth.make_scene(2)
    _run(B, ho, s, cams=s.cameras[:2])


def test_config3_scaled_fp16_exact_path(B, ho, synth):
    # config 3 recipe (clusters + far shell, fp16 tables/weights) with the FMA decoders: lists bit-exact
    s = synth.make_scene(3, n_gaussians=60_000, width=320, height=180, n_cameras=3)
    st = _run(B, ho, s)
    assert 0.3 < st[0]["V"] / s.n < 0.9


def test_config4_scaled_unbounded(B, ho, synth):
    s = synth.make_scene(4, n_gaussians=50_000, width=311, height=206, n_cameras=2)
    _run(B, ho, s)


def test_high_gain_scene_is_sensitive_to_stage2(B, ho, synth):
    # table entries U(-1,1) so that a wrong gather cannot hide inside the image tolerance
    s = synth.make_scene(2, n_gaussians=15_000, width=160, height=128, n_cameras=1, table_amp=1.0)
    st = _run(B, ho, s)
    osc = ho.OracleScene(s)
    raw = ho.stage_query(osc, s.cameras[0], ho.stage_cull(osc, s.cameras[0], 160, 128)[1])
    assert np.abs(raw[:, :8]).std() > 0.05


def test_edge_cases(B, ho, synth):
    import torch
    # (a) nothing visible: camera looks away from everything
    s = synth.tiny_scene(n=32, W=32, H=32)
    s.pos[2, :] = -10.0 - np.abs(s.pos[2, :])          # all behind the first camera (eye z=-3 looking +z)
    st = _run(B, ho, s, cams=s.cameras[:1])
    assert st[0]["V"] == 0 and st[0]["D"] == 0
    # (b) a single Gaussian, 1x1 and 17x1 images
    s = synth.tiny_scene(n=1, W=17, H=1)
    s.pos[:, 0] = 0.0
    _run(B, ho, s, cams=s.cameras[:1])
    s = synth.tiny_scene(n=3, W=1, H=1)
    _run(B, ho, s, cams=s.cameras[:1])
    # (c) huge splats covering every tile (max tiles-touched per Gaussian)
    s = synth.tiny_scene(n=40, W=64, H=48, scale_mean=1.5)
    st = _run(B, ho, s, cams=s.cameras[:1])
    assert st[0]["D"] >= 0.5 * st[0]["V"] * 12
    # (e) fx != fy on a non-square image: limx / limy, the Jacobian and the ray directions each use their own focal length
    s = synth.tiny_scene(n=200, W=80, H=48, seed=21)
    for c in s.cameras:
        c.fy = float(np.float32(2.0 * c.fx))
    _run(B, ho, s)
    # (d) tau_T = 0 composites everywhere; tau_T = 1 nowhere
    for tau in (0.0, 1.0):
        s = synth.tiny_scene(n=48, W=32, H=32)
        s.tau_T = tau
        _run(B, ho, s, cams=s.cameras[:1])


def test_large_tile_grid_takes_radix_route(B, ho, synth):
    # 104 x 100 = 10,400 tiles > the ordered-counting limit: binning falls back to (tile, rank) pairs + radix sort
    s = synth.tiny_scene(n=400, W=1664, H=1600, scale_mean=-3.0)
    s.tau_T = 1.0                                                  # no background pixels: keeps the oracle quick
    st = _run(B, ho, s, cams=s.cameras[:1])
    assert st[0]["D"] > st[0]["V"]


def test_status_codes_on_device(B, synth):
    import ctypes as C
    import torch
    s = synth.tiny_scene(n=16)
    lib = B.load_library()
    d = B.make_desc(s, 32, 32)
    h = C.c_void_p()
    assert lib.hyrf_create_scene(C.byref(d), C.byref(h)) == B.HYRF_OK
    out = torch.zeros(32, 32, 3, device="cuda")
    cam = B.camera_struct(s.cameras[0])
    assert lib.hyrf_render(h, C.byref(cam), 32, 32, C.c_void_p(out.data_ptr())) == B.HYRF_ERR_NOT_READY
    lib.hyrf_destroy_scene(h)
    hs = B.HyrfScene(s)
    with pytest.raises(B.HyrfError) as e:
        hs.render(s.cameras[0], W=64, H=64)                      # beyond max_width
    assert e.value.status == B.HYRF_ERR_INVALID_ARG
    far = synth.look_at(np.array([0.0, 0.0, -150.0]), 32, 32)     # camera outside the background sphere
    with pytest.raises(B.HyrfError) as e:
        hs.render(far)
    assert e.value.status == B.HYRF_ERR_CAMERA
    bad = synth.look_at(np.array([0.0, 0.0, -3.0]), 32, 32)
    bad.fx = float("nan")
    with pytest.raises(B.HyrfError) as e:
        hs.render(bad)
    assert e.value.status == B.HYRF_ERR_CAMERA
    out2 = hs.render(s.cameras[0])                                # still usable after errors
    torch.cuda.synchronize()
    assert torch.isfinite(out2).all()
    host = hs.render_host(s.cameras[0])
    assert (host == out2.cpu()).all()                             # hyrf_render_host = same pass + D2H copy
    hs.close()


def test_render_is_deterministic_and_scratch_grows(B, synth):
    import torch
    s = synth.make_scene(2, n_gaussians=5_000, width=512, height=512, n_cameras=1)
    s.scale_logit[:] = 0.5                                        # big splats: entry count far above the initial guess
    hs = B.HyrfScene(s)
    a = hs.render(s.cameras[0]).clone()
    b = hs.render(s.cameras[0]).clone()
    torch.cuda.synchronize()
    assert (a == b).all()
    hs.debug_enable(0)
    hs.render(s.cameras[0])
    assert int(hs.debug_fetch(B.DBG_COUNTERS)[2]) > 8 * s.n + 65536
    hs.close()


@pytest.mark.parametrize("path", ["MMA", "HMMA", "WS"])
def test_config3_scaled_fp16_tensor_core_path(B, ho, synth, path):
    # both tensor-core kernels (tcgen05 CTA tiles; mma.sync warp tiles): mask bit-exact, raw logits within 2e-3,
    # list symmetric difference reported and bounded, image within 1e-2 (SURVEY §8c H1 protocol)
    s = synth.make_scene(3, n_gaussians=60_000, width=320, height=180, n_cameras=3)
    st = _run(B, ho, s, mlp_path=getattr(B, "HYRF_MLP_" + path), exact=False)
    assert max(x["raw_geo_maxdiff"] for x in st) > 0.0          # really a different arithmetic path
    print("tensor-core path stats:", st[0])


@pytest.mark.parametrize("path", ["MMA", "HMMA", "WS"])
def test_tensor_core_path_high_gain(B, ho, synth, path):
    # large table entries: decoder outputs O(1), so operand layout / K-order mistakes cannot hide in the tolerance
    s = synth.make_scene(3, n_gaussians=20_000, width=160, height=96, n_cameras=1, table_amp=1.0)
    import torch
    hs = B.HyrfScene(s, mlp_path=getattr(B, "HYRF_MLP_" + path))
    hs.debug_enable()
    hs.render(s.cameras[0])
    torch.cuda.synchronize()
    raw = hs.debug_fetch(B.DBG_STAGE2_RAW)
    idx = hs.debug_fetch(B.DBG_VIS_IDX)
    osc = ho.OracleScene(s)
    ref = ho.stage_query(osc, s.cameras[0], idx)
    assert np.abs(ref).max() > 0.3
    err = np.abs(raw - ref)
    assert err.max() < 2e-2 and err.mean() < 1e-3, (err.max(), err.mean())
    hs.close()


def test_config3_full_one_camera_both_paths(B, ho, synth):
    # BASELINE config 3 at full size (1M Gaussians, 1280x720), camera 0: exact path bit-exact lists; tensor paths by
    # hand-off (lists bit-exact given the GPU's attributes); AUTO is the workload and launch configuration bench.py times
    s = synth.make_scene(3, n_cameras=1)
    _run(B, ho, s, mlp_path=B.HYRF_MLP_FMA, exact=True)
    st = _run(B, ho, s, mlp_path=B.HYRF_MLP_AUTO, exact=False, label="config3_full_AUTO")
    print("config 3 full, tcgen05 path:", {k: v for k, v in st[0].items() if not isinstance(v, list)})
    _run(B, ho, s, mlp_path=B.HYRF_MLP_HMMA, exact=False, label="config3_full_HMMA")
    _run(B, ho, s, mlp_path=B.HYRF_MLP_WS, exact=False, label="config3_full_WS")


def test_config4_full_one_camera_both_paths(B, ho, synth):
    # BASELINE config 4 at full size (2M Gaussians, unbounded scene, 1245x825 with ragged tiles), camera 0: the launch
    # configuration bench.py --config 4 times (AUTO -> tensor-core decoders, ordered binning) by hand-off, and the exact
    # path with every list compared bit for bit
    s = synth.make_scene(4, n_cameras=1)
    st = _run(B, ho, s, mlp_path=B.HYRF_MLP_AUTO, exact=False, label="config4_full_AUTO")
    assert st[0]["V"] > 1_000_000
    print("config 4 full, tcgen05 path:", {k: v for k, v in st[0].items() if not isinstance(v, list)})
    _run(B, ho, s, mlp_path=B.HYRF_MLP_FMA, exact=True, label="config4_full_FMA")


def test_config5_points(B, ho, synth):
    # BASELINE config 5: the 500k @ 256x256 point element by element on both paths, and the 500k @ 1920x1080 point
    # (8160 tiles) on the exact path so that its lists are compared bit for bit
    s = synth.make_scene(5, n_gaussians=500_000, width=256, height=256)
    _run(B, ho, s, mlp_path=B.HYRF_MLP_FMA, exact=True)
    _run(B, ho, s, mlp_path=B.HYRF_MLP_AUTO, exact=False)
    s = synth.make_scene(5, n_gaussians=500_000, width=1920, height=1080)
    _run(B, ho, s, mlp_path=B.HYRF_MLP_FMA, exact=True)


def test_config5_500k_at_4k_exact_lists(B, ho, synth):
    # BASELINE config 5, 500k @ 3840x2160 (32,400 tiles, D ~ 57M entries): exact path, every per-tile list bit for bit
    s = synth.make_scene(5, n_gaussians=500_000, width=3840, height=2160)
    st = _run(B, ho, s, mlp_path=B.HYRF_MLP_FMA, exact=True, label="config5_500k_4K_FMA")
    assert st[0]["D"] > 40_000_000


@pytest.mark.parametrize("abl", [1, 2, 4, 8, 1 | 2, 4 | 8, 15])
def test_ablation_switches_exact_path(B, ho, synth, abl):
    # PAPER.md Table 5 switches on the exact path: everything bit-exact against the oracle's
    # same switch; config-3 recipe so that ~40 % of the Gaussians are outside the frustum (NO_CULL has work to do)
    s = synth.make_scene(3, n_gaussians=30_000, width=208, height=120, n_cameras=2)
    st = _run(B, ho, s, ablation=abl)
    if abl & 1:
        assert st[0]["V"] == s.n                      # every stored Gaussian was queried


def test_ablation_switches_tensor_path(B, ho, synth):
    s = synth.make_scene(3, n_gaussians=30_000, width=208, height=120, n_cameras=1)
    for abl in (1, 8, 1 | 2 | 8, 4):
        _run(B, ho, s, mlp_path=B.HYRF_MLP_MMA, exact=(abl & 4) != 0, ablation=abl)
    for abl in (1, 8):
        _run(B, ho, s, mlp_path=B.HYRF_MLP_HMMA, exact=False, ablation=abl)
    for abl in (1, 8, 1 | 2 | 8):
        _run(B, ho, s, mlp_path=B.HYRF_MLP_WS, exact=False, ablation=abl)


def test_sort_overlap_is_schedule_only(B, synth):
    # hyrf_set_sort_overlap: the depth sort beside the field kernel (default) or the frame serialised — same bits out,
    # image and per-tile lists, on both tensor-core kernels and the exact path; several frames so that the second
    # stream's buffers are reused across frames
    import torch
    s = synth.make_scene(3, n_gaussians=80_000, width=320, height=180, n_cameras=4)
    for path in (B.HYRF_MLP_MMA, B.HYRF_MLP_HMMA, B.HYRF_MLP_WS, B.HYRF_MLP_FMA):
        hs = B.HyrfScene(s, mlp_path=path)
        hs.debug_enable()
        ref = []
        hs.set_sort_overlap(False)
        for cam in s.cameras:
            img = hs.render(cam).clone()
            torch.cuda.synchronize()
            ref.append((img, hs.debug_fetch(B.DBG_TILE_LIST).copy(), hs.debug_fetch(B.DBG_TILE_RANGES).copy()))
        hs.set_sort_overlap(True)
        for rep in range(2):
            for cam, (img0, list0, ranges0) in zip(s.cameras, ref):
                img = hs.render(cam)
                torch.cuda.synchronize()
                assert torch.equal(img, img0)
                assert np.array_equal(hs.debug_fetch(B.DBG_TILE_RANGES), ranges0)
                assert np.array_equal(hs.debug_fetch(B.DBG_TILE_LIST), list0)
        hs.close()


def test_no_cull_image_equals_full_model(B, synth):
    # NO_CULL moves work, not pixels: same image bit for bit on the exact path
    import torch
    s = synth.make_scene(3, n_gaussians=30_000, width=208, height=120, n_cameras=1)
    hs = B.HyrfScene(s, mlp_path=B.HYRF_MLP_FMA)
    a = hs.render(s.cameras[0]).clone()
    hs.set_ablation(B.ABL_NO_CULL)
    b = hs.render(s.cameras[0]).clone()
    torch.cuda.synchronize()
    assert (a == b).all()
    with pytest.raises(B.HyrfError):
        hs.set_ablation(16)
    hs.close()


@pytest.mark.parametrize("n,w,h", [(40_000, 320, 180), (400_000, 1280, 720)])
def test_pipelined_frames_match_serial_ones(B, synth, n, w, h):
    # A stream of frames (hyrf_render_host_async): frame k+1's cull and depth sort run beside frame k's rasterizer on
    # double-buffered scratch, the field kernel takes every SM, the copies ride a third stream. Every delivered image
    # must be, bit for bit, the image of the one-frame-at-a-time call; 3 passes over 7 cameras so that both buffer sets
    # are reused many times, interleaved with a serial frame in between (mode switches mid-stream).
    import torch
    s = synth.make_scene(3, n_gaussians=n, width=w, height=h, n_cameras=7)
    hs = B.HyrfScene(s)
    ref = [hs.render_host(c).clone() for c in s.cameras]
    bufs = [torch.empty((h, w, 3), dtype=torch.float32).pin_memory() for _ in range(2)]
    cs = [B.camera_struct(c) for c in s.cameras]
    pending = []          # (frame index, buffer index)
    k = 0
    for rep in range(3):
        for i in range(len(cs)):
            if len(pending) == 2:                     # the buffer about to be reused holds the oldest frame
                hs.host_sync()
                for (fi, bi) in pending:
                    assert (bufs[bi] == ref[fi]).all(), f"pipelined frame {fi} (pass {rep}) differs"
                pending = []
            hs.render_host_async(cs[i], w, h, bufs[k & 1])
            pending.append((i, k & 1))
            k += 1
        hs.host_sync()
        for (fi, bi) in pending:
            assert (bufs[bi] == ref[fi]).all()
        pending = []
        assert (hs.render_host(s.cameras[rep]) == ref[rep]).all()     # a serial frame between two pipelined runs
    hs.close()


def test_pipelined_host_delivery_matches_synchronous(B, synth):
    # hyrf_render_host_async: two frames in flight, copies on a second stream; every delivered image must be the
    # image the synchronous call produces for the same camera
    import torch
    s = synth.make_scene(3, n_gaussians=40_000, width=320, height=180, n_cameras=5)
    hs = B.HyrfScene(s)
    ref = [hs.render_host(c).clone() for c in s.cameras]
    bufs = [torch.empty((180, 320, 3), dtype=torch.float32).pin_memory() for _ in range(2)]
    got = []
    for i, c in enumerate(s.cameras):
        if i >= 2:
            hs.host_sync()                      # buffer i & 1 is about to be reused
            got.append(bufs[i & 1].clone())
        hs.render_host_async(B.camera_struct(c), 320, 180, bufs[i & 1])
    hs.host_sync()
    # frames 0..2 were cloned when their buffer came up for reuse; the last two are still in the buffers
    got.append(bufs[1].clone() if len(s.cameras) % 2 == 0 else bufs[(len(s.cameras) - 2) & 1].clone())
    got.append(bufs[(len(s.cameras) - 1) & 1].clone())
    assert len(got) == len(ref)
    for i, (a, b) in enumerate(zip(got, ref)):
        assert (a == b).all(), f"frame {i} differs"
    hs.close()


def test_quantised_tables_exact_path(B, ho, synth):
    # compressed model (PAPER.md:227-229 (3)): 8-bit min-max tables decoded inside the gather.
    # CUDA-core decoders: everything bit-exact against the oracle's same decode
    s = synth.quantize8(synth.make_scene(3, n_gaussians=40_000, width=320, height=180, n_cameras=2, table_amp=0.5))
    st = _run(B, ho, s)
    assert st[0]["D"] > 0
    t = synth.quantize8(synth.tiny_scene(n=64, W=48, H=40, seed=3))        # run-time-shaped kernels
    _run(B, ho, t)


def test_quantised_tables_tensor_path(B, ho, synth):
    # interleaved 4-byte entries (geo c0 c1 | app c0 c1) on the tcgen05 path; high-gain tables so that a wrong
    # (min, step) or a swapped field cannot hide in the tolerance
    import torch
    s = synth.quantize8(synth.make_scene(3, n_gaussians=40_000, width=320, height=180, n_cameras=2))
    _run(B, ho, s, mlp_path=B.HYRF_MLP_AUTO, exact=False)
    s = synth.quantize8(synth.make_scene(3, n_gaussians=20_000, width=160, height=96, n_cameras=1, table_amp=1.0))
    for path in (B.HYRF_MLP_MMA, B.HYRF_MLP_HMMA, B.HYRF_MLP_WS):
        hs = B.HyrfScene(s, mlp_path=path)
        hs.debug_enable()
        hs.render(s.cameras[0])
        torch.cuda.synchronize()
        raw = hs.debug_fetch(B.DBG_STAGE2_RAW)
        ref = ho.stage_query(ho.OracleScene(s), s.cameras[0], hs.debug_fetch(B.DBG_VIS_IDX))
        assert np.abs(ref).max() > 0.3
        err = np.abs(raw - ref)
        assert err.max() < 2e-2 and err.mean() < 1e-3, (path, err.max(), err.mean())
        hs.close()


def _decoded_rows(ho, rvq):
    d = ho.decode_explicit(rvq)
    return np.concatenate([d["pos"], d["scale_logit"][None], d["opacity_logit"][None], d["rgb_logit"]])


@pytest.mark.parametrize("n,stages,K,host", [(4096, 6, 64, False), (4099, 3, 17, True), (1, 1, 1, True),
                                             (50_000, 2, 4096, False), (30_001, 16, 5, False)])
def test_explicit_rvq_decode_bit_exact(B, ho, synth, n, stages, K, host):
    # compressed explicit Gaussians (PAPER.md:227-229 (1)-(2)): the decode kernel against the
    # oracle's decode, bit for bit: vectorised (n % 4 == 0) and scalar (ragged n) variants, codebooks in shared memory
    # and beyond 48 KB (2 x 4096 x 20 B), host and device sources, the 16-stage maximum, a single Gaussian
    s = synth.compress_explicit(synth.make_scene(1, n_gaussians=n, n_cameras=1), stages=stages, codebook_size=K, seed=n)
    if stages == 16:                                   # make the order of the additions matter in every row
        s.explicit_rvq.codebooks[0] += np.float32(1e6)
        s.explicit_rvq.codebooks[1] -= np.float32(1e6)
    hs = B.HyrfScene(s, host_upload=host)
    got = hs.explicit_params()
    want = _decoded_rows(ho, s.explicit_rvq)
    assert (got.view(np.uint32) == want.view(np.uint32)).all()
    assert hs.last_decode_time() > 0.0
    hs.close()


def test_explicit_rvq_every_half_pattern_and_rejection(B, ho, synth):
    import copy
    base = synth.make_scene(1, n_gaussians=63488, n_cameras=1)           # 63488 = number of finite binary16 patterns
    s = synth.compress_explicit(base, stages=2, codebook_size=8)
    bits = np.arange(65536, dtype=np.uint16)
    bits = bits[(bits & 0x7C00) != 0x7C00]
    s.explicit_rvq.pos_h = np.stack([bits, bits[::-1], np.roll(bits, 7)])
    hs = B.HyrfScene(s)
    got = hs.explicit_params()
    assert (got.view(np.uint32) == _decoded_rows(ho, s.explicit_rvq).view(np.uint32)).all()
    # a code outside the codebook is refused, names its Gaussian, and leaves the scene not renderable
    bad = copy.copy(s.explicit_rvq)
    bad.codes = s.explicit_rvq.codes.copy()
    bad.codes[1, 12345] = 8
    bad.codes[0, 40000] = 9
    with pytest.raises(B.HyrfError) as e:
        hs.upload_explicit_rvq(bad)
    assert e.value.status == B.HYRF_ERR_INVALID_ARG and "12345" in str(e.value)
    with pytest.raises(B.HyrfError) as e:
        hs.render(base.cameras[0])
    assert e.value.status == B.HYRF_ERR_NOT_READY
    hs.upload_explicit_rvq(s.explicit_rvq)                                # and recovers with a valid upload
    assert (hs.explicit_params().view(np.uint32) == got.view(np.uint32)).all()
    hs.close()


def test_compressed_model_render_exact_path(B, ho, synth):
    # the whole compressed model of PAPER.md:227-229: binary16 positions + R-VQ properties + 8-bit tables, rendered
    # through the exact decoders: every stage bit-exact against the oracle rendering the same compressed scene
    s = synth.make_scene(3, n_gaussians=40_000, width=320, height=180, n_cameras=2, table_amp=0.5)
    st = _run(B, ho, synth.compress_explicit(synth.quantize8(s)))
    assert st[0]["D"] > 0
    _run(B, ho, synth.compress_explicit(synth.tiny_scene(n=61, W=48, H=40, seed=5), stages=4, codebook_size=16))
    _run(B, ho, synth.compress_explicit(synth.make_scene(2, n_gaussians=20_000, width=200, height=136, n_cameras=2)))


def test_compressed_model_render_tensor_path(B, ho, synth):
    s = synth.compress_explicit(synth.quantize8(synth.make_scene(3, n_gaussians=40_000, width=320, height=180, n_cameras=2)))
    _run(B, ho, s, mlp_path=B.HYRF_MLP_AUTO, exact=False)


def test_fields_then_explicit_upload_order(B, ho, synth):
    # plain explicit arrays first, then replaced by the compressed ones: the render follows the last upload
    import torch
    plain = synth.tiny_scene(n=64, W=32, H=32)
    comp = synth.compress_explicit(plain, stages=2, codebook_size=4)
    hs = B.HyrfScene(plain)
    a = hs.render(plain.cameras[0]).cpu().numpy()
    hs.upload_explicit_rvq(comp.explicit_rvq)
    b = hs.render(plain.cameras[0]).cpu().numpy()
    torch.cuda.synchronize()
    assert not (a == b).all()
    want = ho.render(ho.OracleScene(comp), comp.cameras[0])["out"]
    assert np.abs(b - want).mean() <= 1e-4 and (np.abs(b - want) <= 2e-3).mean() > 0.99
    hs.upload(plain)                                                       # and back
    assert (hs.render(plain.cameras[0]).cpu().numpy() == a).all()
    hs.close()


@pytest.mark.parametrize("n,W,H", [(4_000_000, 3840, 2160), (4_000_000, 1920, 1080), (4_000_000, 256, 256)])
def test_config5_4m_points_sampled(B, ho, synth, n, W, H):
    # BASELINE config 5's largest point (4M Gaussians at 3840x2160, D ~ 4e8 tile entries) in the launch configuration
    # bench.py --config 5 times (AUTO decoders, macro-tile binning, per-tile lists NOT materialised). The oracle cannot
    # bin 4e8 entries in seconds, so: cull element by element; stages 2-4a on 4096 sampled Gaussians; stages 4b-5 on
    # 24 sampled tiles whose depth-ordered lists are rebuilt one by one from the exported records (hand-off)
    # and rasterised by the oracle; stage 6 on the whole image from the exported (C_fg, T); properties everywhere.
    # (the 1080p and 256x256 points of the 4M row go through the same protocol)
    import torch
    s = synth.make_scene(5, n_gaussians=n, width=W, height=H)
    cam = s.cameras[0]
    hs = B.HyrfScene(s, mlp_path=B.HYRF_MLP_AUTO)
    hs.debug_enable(B.DBG_ALL & ~((1 << B.DBG_TILE_LIST) | (1 << B.DBG_TILE_RANGES)))
    out = hs.render(cam)
    torch.cuda.synchronize()
    out = out.cpu().numpy()
    osc = ho.OracleScene(s)
    mask, vis = ho.stage_cull(osc, cam, W, H)
    assert (hs.debug_fetch(B.DBG_VIS_MASK) == mask).all()
    assert (hs.debug_fetch(B.DBG_VIS_IDX) == vis).all()
    V = len(vis)
    assert V > 3_000_000
    proj, rect = hs.debug_fetch(B.DBG_PROJ), hs.debug_fetch(B.DBG_RECT)
    cnt = hs.debug_fetch(B.DBG_COUNTERS)
    r64 = rect.astype(np.int64)
    tiles = np.where((r64[:, 1] > r64[:, 0]) & (r64[:, 3] > r64[:, 2]), (r64[:, 1] - r64[:, 0]) * (r64[:, 3] - r64[:, 2]), 0)
    assert int(cnt[1]) == V and int(cnt[2]) == int(tiles.sum())
    # stages 2-4a on a sample
    rng = np.random.default_rng(5)
    pick = np.sort(rng.choice(V, 4096, replace=False))
    raw_o = ho.stage_query(osc, cam, vis[pick])
    at_o = ho.stage_aggregate(osc, vis[pick], raw_o)
    pr_o = ho.stage_project(osc, cam, W, H, vis[pick], at_o)
    assert np.abs(hs.debug_fetch(B.DBG_STAGE2_RAW)[pick] - raw_o).max() <= 2e-3
    assert np.abs(hs.debug_fetch(B.DBG_STAGE3_ATTRS)[pick] - at_o).max() <= 2e-3
    live = pr_o["tiles"] > 0
    assert (proj[pick][live][:, :3].view(np.uint32) == pr_o["proj"][live][:, :3].view(np.uint32)).all()   # u, v, depth: no field input
    assert np.allclose(proj[pick][live][:, 3:], pr_o["proj"][live][:, 3:], rtol=5e-3, atol=2e-3)
    assert (rect[pick] == pr_o["rect"]).mean() > 0.995           # a rectangle edge can move by one tile under 1e-4 noise
    # stages 4b-5 on sampled tiles (hand-off from the exported records)
    gx, gy = (W + 15) // 16, (H + 15) // 16
    depth_bits = np.ascontiguousarray(proj[:, 2]).view(np.uint32)
    ranges = np.zeros((gx * gy, 2), np.uint32)
    lists, pos, sampled = [], 0, []
    cx, cy = gx // 2, gy // 2
    n_rand = 19 if W > 1000 else 3            # 256 x 256: every tile holds ~10^5 entries of the 4M scene
    cand = [(cx, cy), (max(cx - 7, 0), min(cy + 3, gy - 1)), (0, 0), (gx - 1, gy - 1), (gx - 1, 0)] + \
           [(int(rng.integers(gx // 4, 3 * gx // 4)), int(rng.integers(gy // 4, 3 * gy // 4))) for _ in range(n_rand)]
    for tx, ty in cand:
        t = ty * gx + tx
        if t in sampled:
            continue
        mem = np.nonzero((tiles > 0) & (rect[:, 0] <= tx) & (tx < rect[:, 1]) & (rect[:, 2] <= ty) & (ty < rect[:, 3]))[0]
        mem = mem[np.argsort(depth_bits[mem], kind="stable")]        # ranks ascend with ids: ties fall to the id
        ranges[t] = (pos, pos + len(mem))
        lists.append(mem.astype(np.uint32))
        pos += len(mem)
        sampled.append(t)
    assert pos > 10_000
    rs = ho.stage_raster(W, H, proj, np.concatenate(lists), ranges)
    fg, T = hs.debug_fetch(B.DBG_FG).reshape(H, W, 3), hs.debug_fetch(B.DBG_FINAL_T).reshape(H, W)
    assert np.isfinite(out).all() and (T >= 0).all() and (T <= 1).all()
    n_px = n_fragile = 0
    for t in sampled:
        ty, tx = divmod(t, gx)
        sl = (slice(ty * 16, min(ty * 16 + 16, H)), slice(tx * 16, min(tx * 16 + 16, W)))
        fragile = (rs["m_alpha"][sl] < 5e-8) | (rs["m_stop"][sl] < 5e-5)
        d = np.abs(fg[sl] - rs["cfg"][sl]).max(axis=-1)
        dT = np.abs(T[sl] - rs["T"][sl])
        assert d[~fragile].max(initial=0.0) <= 2e-3 and dT[~fragile].max(initial=0.0) <= 2e-3, (tx, ty, d.max(), dT.max())
        assert d.max() <= 2e-3 + 1.0 / 255.0 + 1e-2
        n_px += fragile.size
        n_fragile += int(fragile.sum())
    assert n_fragile < 0.01 * n_px
    # stage 6 on the whole image, from the exported foreground and transmittance
    want, bgm = ho.stage_background(osc, cam, W, H, fg, T)
    near_tau = np.abs(T - np.float32(s.tau_T)) < 1e-5
    assert (hs.debug_fetch(B.DBG_BG_MASK).reshape(H, W).astype(bool)[~near_tau] == bgm.astype(bool)[~near_tau]).all()
    assert np.abs(out - want)[~near_tau].max() <= 1e-2
    assert np.abs(out - want)[~near_tau].mean() <= 1e-4
    hs.close()


@pytest.mark.parametrize("mode", [1, 2, 3, 4])
def test_both_rasterizers_against_the_oracle(B, ho, synth, mode):
    # hyrf_set_raster_mode: 1 = every warp blends every staged entry (raster.cu), 2 = per-warp lists over 8 x 4 pixel
    # blocks (raster_warp.cu). Each against the oracle on its own: small splats (config 3 recipe), large splats at a
    # ragged resolution (tiny scene, scale_mean -1: blocks outside the image, every block reached), per-tile lists
    # (<= 1024 tiles) and macro-tile lists (> 1024 tiles)
    _run(B, ho, synth.make_scene(3, n_gaussians=60_000, width=320, height=180, n_cameras=2), raster_mode=mode)
    _run(B, ho, synth.make_scene(3, n_gaussians=30_000, width=640, height=360, n_cameras=1), raster_mode=mode)
    _run(B, ho, synth.tiny_scene(n=64, W=45, H=37, seed=9, scale_mean=-1.0), raster_mode=mode)
    _run(B, ho, synth.make_scene(2, n_gaussians=20_000, width=200, height=136, n_cameras=2), raster_mode=mode)


def test_rasterizer_choice_changes_no_bit(B, synth):
    import torch
    s = synth.make_scene(3, n_gaussians=200_000, width=640, height=360, n_cameras=2)
    hs = B.HyrfScene(s)
    outs = {}
    for mode in (1, 2, 3, 4, 0):
        hs.set_raster_mode(mode)
        frames = []
        for cam in s.cameras:
            o = hs.render(cam)
            torch.cuda.synchronize()
            frames.append((o.cpu().numpy().copy(), hs.debug_fetch(B.DBG_FINAL_T).copy()))
        outs[mode] = frames
    for mode in (2, 3, 4, 0):
        for (a, ta), (b, tb) in zip(outs[1], outs[mode]):
            assert (a.view(np.uint32) == b.view(np.uint32)).all() and (ta.view(np.uint32) == tb.view(np.uint32)).all()
    hs.set_raster_mode(1); hs.render(s.cameras[0]); assert hs.last_raster_mode() == 1
    hs.set_raster_mode(2); hs.render(s.cameras[0]); assert hs.last_raster_mode() == 2
    hs.set_raster_mode(3); hs.render(s.cameras[0]); assert hs.last_raster_mode() == 3
    hs.set_raster_mode(4); hs.render(s.cameras[0]); assert hs.last_raster_mode() == 4
    with pytest.raises(B.HyrfError) as e:
        hs.set_raster_mode(5)
    assert e.value.status == B.HYRF_ERR_INVALID_ARG
    hs.close()


def _backward_case(B, ho, scene, cam, seed=0):
    import torch
    hs = B.HyrfScene(scene, mlp_path=B.HYRF_MLP_FMA)
    hs.debug_enable()
    hs.render(cam)
    torch.cuda.synchronize()
    orc = ho.render(ho.OracleScene(scene), cam)
    W, H, V = cam.W, cam.H, len(orc["vis_idx"])
    assert (hs.debug_fetch(B.DBG_TILE_LIST) == orc["list_id"]).all()      # same lists, same records: same frozen set
    rng = np.random.default_rng(seed)
    gc = rng.normal(0, 1, (H, W, 3)).astype(np.float32)
    gt = rng.normal(0, 1, (H, W)).astype(np.float32)
    got = hs.raster_backward(torch.from_numpy(gc).cuda(), torch.from_numpy(gt).cuda(), V)
    torch.cuda.synchronize()
    got = got.cpu().numpy().astype(np.float64)
    want = ho.stage_raster_backward(W, H, orc["proj"], orc["list_rank"], orc["ranges"], gc, gt)
    hs.close()
    return got, want, orc


@pytest.mark.parametrize("case", ["tiny", "tiny_big_splats", "config1", "config3_scaled", "config3_full"])
def test_raster_backward_against_oracle(B, ho, synth, case):
    # hyrf_raster_backward (DESIGN.md §2 D12, first piece) against the oracle's float64 backward
    # on the same frozen decisions. fp32 sums in atomic order + T recovered by division: tolerance 2e-3 of each
    # column's scale plus 2e-3 relative; a pair whose decision sits on the ex2.approx / exp difference may flip for a
    # pixel or two, which stays inside that bound.
    if case == "tiny":
        s = synth.tiny_scene(n=48, W=32, H=32)
    elif case == "tiny_big_splats":
        s = synth.tiny_scene(n=64, W=45, H=37, seed=9, scale_mean=-1.0)      # ragged tiles, deep lists, clamped alphas
    elif case == "config1":
        s = synth.make_scene(1)
    elif case == "config3_scaled":
        s = synth.make_scene(3, n_gaussians=60_000, width=320, height=180, n_cameras=1)
    else:
        s = synth.make_scene(3, n_cameras=1)          # BASELINE config 3 at full size: what bench.py --backward times
    got, want, orc = _backward_case(B, ho, s, s.cameras[0], seed=len(case))
    assert np.isfinite(got).all()
    scale = np.abs(want).max(axis=0)
    assert (scale > 0).all()
    err = np.abs(got - want)
    assert (err <= 2e-3 * scale + 2e-3 * np.abs(want)).all(), (err.max(axis=0) / scale)
    untouched = orc["tiles"] == 0
    assert (got[untouched] == 0).all()                                       # a Gaussian in no list gets no gradient


def test_raster_backward_needs_the_lists(B, synth):
    import torch
    s = synth.tiny_scene(n=16)
    hs = B.HyrfScene(s)
    hs.render(s.cameras[0])
    z = torch.zeros(32, 32, 3, device="cuda")
    with pytest.raises(B.HyrfError) as e:
        hs.raster_backward(z, z[..., 0], 16)
    assert e.value.status == B.HYRF_ERR_NOT_READY
    hs.close()


def _adversarial_scene(synth, n=600, W=1280, H=720, seed=31):
    # Long thin splats for the reach tests of csrc/raster_common.cuh (VERDICT r1 finding 4): config-2 recipe with
    # high-gain tables and the geometry decoder's output rows scaled so that s_n spreads over +-5 logits around
    # s_e = 0: scales sigma(-5) .. sigma(5) = 0.0067 .. 0.993 world units -> anisotropy up to 150:1, splats hundreds of
    # pixels long and a few pixels wide at random orientations (r_n is as random as s_n); opacity logits N(-2.5, 2.5)
    # put many peak alphas near the 1/255 threshold. 3600 tiles -> macro-tile lists.
    s = synth.make_scene(2, n_gaussians=n, width=W, height=H, n_cameras=1, table_amp=1.0, seed=seed)
    rng = np.random.default_rng(seed)
    s.scale_logit[:] = rng.normal(0.0, 0.5, n).astype(np.float32)
    s.opacity_logit[:] = rng.normal(-2.5, 2.5, n).astype(np.float32)
    w = s.geo_w.copy()
    m = s.geo_mlp
    off = m.in_dim * m.hidden + (m.n_hidden - 1) * m.hidden * m.hidden
    out = w[off:].reshape(m.out_dim, m.hidden)
    out[1:4] *= 40.0          # rows of s_n
    out[4:8] *= 10.0          # rows of r_n
    s.geo_w = w
    s.cameras = [synth.look_at(np.array([0.3, 0.2, -3.0]), W, H)]
    s.name = f"adversarial_n{n}_{W}x{H}"
    return s


def test_adversarial_long_thin_splats(B, ho, synth):
    import torch
    s = _adversarial_scene(synth)
    osc = ho.OracleScene(s)
    cam = s.cameras[0]
    orc = ho.render(osc, cam)
    # the scene really is adversarial: anisotropy >= 100:1 and splats >= 500 px long, peak alphas around the threshold
    sc = orc["attrs"][:, :3]
    assert (sc.max(axis=1) / sc.min(axis=1)).max() >= 100.0
    assert orc["radius"].max() >= 250.0                       # 3 sigma on each side
    live = orc["tiles"] > 0
    assert (np.abs(orc["proj"][live][:, 6] - 1.0 / 255.0) < 2e-3).sum() >= 5
    outs = {}
    for mode in (1, 2, 3, 4):
        st = _run(B, ho, s, raster_mode=mode, label=f"adversarial_mode{mode}")
        assert st[0]["D"] > 50 * st[0]["V"]
        hs = B.HyrfScene(s, mlp_path=B.HYRF_MLP_FMA)
        hs.set_raster_mode(mode)
        o = hs.render(cam)
        torch.cuda.synchronize()
        outs[mode] = (o.cpu().numpy().copy(), hs.debug_fetch(B.DBG_FINAL_T).copy())
        hs.close()
    for mode in (2, 3, 4):
        assert (outs[1][0].view(np.uint32) == outs[mode][0].view(np.uint32)).all()
        assert (outs[1][1].view(np.uint32) == outs[mode][1].view(np.uint32)).all()
    # and at a ragged small resolution with per-tile lists (<= 1024 tiles)
    s2 = _adversarial_scene(synth, n=200, W=333, H=250, seed=32)
    for mode in (1, 2, 3, 4):
        _run(B, ho, s2, raster_mode=mode, label=f"adversarial_small_mode{mode}")


def test_single_shared_field(B, ho, synth):
    # PAPER.md:233, Table 5 "w/o Decouple": one field for all properties. The pass has no switch for it: the SAME table
    # is uploaded as the geometry and the appearance field (hyrf.h hyrf_set_ablation). Oracle vs GPU on every decoder
    # path; high-gain entries so that reading the wrong half of an interleaved entry cannot hide.
    s = synth.make_scene(3, n_gaussians=30_000, width=320, height=180, n_cameras=2, table_amp=1.0)
    s.app_table = s.geo_table
    _run(B, ho, s, mlp_path=B.HYRF_MLP_FMA, exact=True, label="shared_field_FMA")
    for path in ("MMA", "HMMA", "WS"):
        st = _run(B, ho, s, mlp_path=getattr(B, "HYRF_MLP_" + path), exact=False, label="shared_field_" + path)
        assert st[0]["raw_geo_maxdiff"] > 0.0
    t = synth.tiny_scene(n=64, W=48, H=40, seed=13)           # run-time-shaped kernels, fp32
    t.app_table = t.geo_table
    _run(B, ho, t, label="shared_field_tiny")


class _GuardAllocator:
    """hyrf_scene_desc.alloc backed by torch, with a canary-filled guard band on both sides of every allocation."""
    GUARD = 1 << 16

    def __init__(self, torch):
        self.torch, self.live = torch, {}

    def alloc(self, nbytes):
        t = self.torch.full((nbytes + 2 * self.GUARD,), 0xA5, dtype=self.torch.uint8, device="cuda")
        self.live[t.data_ptr() + self.GUARD] = (t, nbytes)
        return t.data_ptr() + self.GUARD

    def release(self, ptr):
        self.check_one(ptr)
        del self.live[ptr]

    def check_one(self, ptr):
        t, nbytes = self.live[ptr]
        assert bool((t[:self.GUARD] == 0xA5).all()), "write below an allocation"
        assert bool((t[self.GUARD + nbytes:] == 0xA5).all()), f"write beyond an allocation of {nbytes} bytes"

    def check(self):
        self.torch.cuda.synchronize()
        for p in list(self.live):
            self.check_one(p)


def test_list_export_beyond_initial_capacity_stays_in_bounds(B, ho, synth):
    # with the per-tile lists exported and D above the scratch's first size, the rasterizer wrote the
    # lists past the pair buffer before the host grew it. Every library allocation sits between canary bands here.
    import torch
    s = synth.make_scene(3, n_gaussians=20_000, width=640, height=360, n_cameras=1)     # 920 tiles -> per-tile lists
    s.scale_logit[:] = -1.0                                     # big splats: D far above 4 N + 65536
    for (W, H) in ((640, 360), (1280, 720)):                    # per-tile lists, then macro-tile lists (3600 tiles)
        s.cameras = [synth.look_at(np.array([4.0, 0.0, 0.0]), W, H)]
        ga = _GuardAllocator(torch)
        hs = B.HyrfScene(s, mlp_path=B.HYRF_MLP_FMA, allocator=ga)
        hs.debug_enable()
        out = hs.render(s.cameras[0])
        ga.check()
        cnt = hs.debug_fetch(B.DBG_COUNTERS)
        assert int(cnt[2]) > 4 * s.n + 65536 + (4 * s.n + 65536) // 4 + 4096      # above the first capacity
        gpu = hs.debug_all(W, H)
        orc = ho.render(ho.OracleScene(s), s.cameras[0])
        compare_frame(orc, gpu, out.cpu().numpy(), s.tau_T, fp16=True, label=f"guarded_{W}x{H}")
        hs.debug_enable(0)                                      # and the blind path: re-binned after growing
        hs.render(s.cameras[0])
        ga.check()
        hs.close()
        torch.cuda.synchronize()
        assert not ga.live


def test_screen_strips_equal_the_whole_image(B, synth):
    # a device bins, rasterises and composites only its strip of tile rows; the rows it writes
    # must be the same bits as in the whole-image render, for macro-tile lists (1280x720, ragged last tile row at 720 =
    # 45 tiles) and per-tile lists (<= 1024 tiles), on the exact and the tensor-core path, for 2, 3 and 5 strips (5 strips
    # of 720 rows: the last rank's strip is empty); rows outside a strip stay untouched
    import torch
    for (n, W, H, path) in ((150_000, 1280, 720, B.HYRF_MLP_AUTO), (40_000, 400, 300, B.HYRF_MLP_FMA)):
        s = synth.make_scene(3, n_gaussians=n, width=W, height=H, n_cameras=2)
        hs = B.HyrfScene(s, mlp_path=path)
        for cam in s.cameras:
            full = hs.render(cam).clone()
            torch.cuda.synchronize()
            for world in (2, 3, 5):
                got = torch.full((H, W, 3), -7.0, device="cuda")
                covered = 0
                for rank in range(world):
                    y0, y1 = synth.strip_rows(H, rank, world)
                    if y0 == y1:
                        continue
                    hs.set_strip(y0, y1)
                    part = torch.full((H, W, 3), -7.0, device="cuda")
                    hs.render(cam, out=part)
                    torch.cuda.synchronize()
                    assert (part[:y0] == -7.0).all() and (part[y1:] == -7.0).all()      # other devices' rows untouched
                    got[y0:y1] = part[y0:y1]
                    covered += y1 - y0
                assert covered == H
                assert torch.equal(got, full), f"strips of {world} differ from the whole image"
            hs.set_strip(0, 0)
            assert torch.equal(hs.render(cam), full)
        with pytest.raises(B.HyrfError) as e:
            hs.set_strip(8, 64)
            hs.render(s.cameras[0])
        assert e.value.status == B.HYRF_ERR_INVALID_ARG
        hs.close()


def _grad_close(got, want, name, rel=2e-2, floor=2e-3):
    # binary32 sums in atomic order against float64: every entry within `floor` of the array's largest magnitude plus
    # `rel` of its own value
    scale = np.abs(want).max()
    err = np.abs(got - want)
    assert np.isfinite(got).all(), name
    assert (err <= floor * scale + rel * np.abs(want)).all(), (name, float(err.max()), float(scale))


@pytest.mark.parametrize("case", ["tiny", "tiny_fp16", "cfg2_scaled", "cfg3_scaled"])
def test_backward_against_oracle(B, ho, synth, case):
    # hyrf_loss_l1_ssim + hyrf_backward (DESIGN.md §2 D13) against oracle/hyrf_oracle_backward.py:
    # the loss value and dL/d image, then every parameter gradient of one camera's training step. Exact decoders, so the
    # frozen decisions (lists, blended prefixes, background mask) coincide with the oracle's binary32 forward.
    import torch
    from oracle import hyrf_oracle_backward as hb
    if case == "tiny":
        s = synth.tiny_scene(n=48, W=32, H=32, table_amp=1.0)
    elif case == "tiny_fp16":
        s = synth.tiny_scene(n=64, W=45, H=37, seed=9, fp16=True, table_amp=1.0)
    elif case == "cfg2_scaled":
        s = synth.make_scene(2, n_gaussians=3000, width=96, height=80, n_cameras=1, table_amp=0.5)
    else:
        s = synth.make_scene(3, n_gaussians=20_000, width=160, height=96, n_cameras=1, table_amp=0.5)
    cam = s.cameras[0]
    rng = np.random.default_rng(len(case))
    gt = rng.uniform(0, 1, (cam.H, cam.W, 3)).astype(np.float32)
    hs = B.HyrfScene(s, mlp_path=B.HYRF_MLP_FMA)
    hs.debug_enable()
    out = hs.render(cam)
    torch.cuda.synchronize()
    fwd = ho.render(ho.OracleScene(s), cam)
    assert (hs.debug_fetch(B.DBG_TILE_LIST) == fwd["list_id"]).all()
    # loss (on the oracle's image, so that both sides differentiate at the same point)
    img = torch.from_numpy(fwd["out"]).cuda()
    L, g_img = hs.loss_l1_ssim(img, torch.from_numpy(gt).cuda(), 0.2)
    L_o, g_o = hb.loss_and_grad(fwd["out"], gt, 0.2)
    assert abs(L - L_o) <= 1e-5 * abs(L_o)
    _grad_close(g_img.cpu().numpy().astype(np.float64), g_o, "dL/d image", rel=1e-3, floor=1e-4)
    # the whole backward from the oracle's image gradient
    want = hb.backward_from_image_grad(s, cam, g_o, fwd=fwd)
    got = hs.backward(torch.from_numpy(g_o.astype(np.float32)).cuda())
    torch.cuda.synchronize()
    for k in ("opacity_logit", "rgb_logit", "scale_logit", "pos", "geo_w", "app_w", "bg_w", "geo_table", "app_table", "bg_table"):
        # fp16 configs: the forward pass rounds features and hidden activations to binary16 (2^-11 relative each), which the
        # float64 oracle treats as the identity: the floor widens from 2e-3 to 5e-3 of the array's largest magnitude
        _grad_close(got[k].cpu().numpy().astype(np.float64), want[k], f"{case}: {k}", floor=5e-3 if s.fp16 else 2e-3)
    # gradients accumulate (hyrf.h: ADDED to what the arrays hold)
    again = hs.backward(torch.from_numpy(g_o.astype(np.float32)).cuda(), grads={k: v.clone() for k, v in got.items()})
    torch.cuda.synchronize()
    assert torch.allclose(again["opacity_logit"], 2 * got["opacity_logit"], rtol=1e-4, atol=1e-9)
    hs.close()


@pytest.mark.gpu
@pytest.mark.parametrize("raster_mode", [1, 2, 3, 4])
def test_retained_lists_give_the_export_paths_gradients(B, synth, raster_mode):
    # hyrf_set_retain_lists: the training switch keeps per-tile lists only up to the entry at which a
    # tile's pixels had all terminated and leaves the rasterizer its early exit. Image: bit-identical. Gradients: those
    # of the debug-export path (whole lists, no early exit) up to the order of the fp32 atomics.
    import torch
    s = synth.make_scene(3, n_gaussians=20_000, width=160, height=96, n_cameras=1, table_amp=0.5)
    s.opacity_logit[:] += 3.0   # opaque enough for tiles to terminate early: the retained lists are really shorter
    cam = s.cameras[0]
    g = torch.from_numpy(np.random.default_rng(3).normal(0, 1, (cam.H, cam.W, 3)).astype(np.float32)).cuda()
    res = {}
    for how in ("export", "retain"):
        hs = B.HyrfScene(s, mlp_path=B.HYRF_MLP_FMA)
        hs.set_raster_mode(raster_mode)
        if how == "export":
            hs.debug_enable((1 << B.DBG_TILE_LIST) | (1 << B.DBG_TILE_RANGES))
        else:
            hs.set_retain_lists(True)
        img = hs.render(cam).clone()
        grads = hs.backward(g)
        torch.cuda.synchronize()
        V = int(hs.debug_fetch(B.DBG_COUNTERS)[1])   # (N, V, D, tiles, Dm)
        with pytest.raises(B.HyrfError) as e:   # a gradient buffer smaller than V is refused
            B._check(hs.lib.hyrf_raster_backward(hs.handle, g.data_ptr(), g[..., 0].contiguous().data_ptr(),
                                                 g.data_ptr(), max(V - 1, 0)))
        assert e.value.status == B.HYRF_ERR_INVALID_ARG
        res[how] = (img, {k: v.clone() for k, v in grads.items()})
        hs.close()
    assert torch.equal(res["export"][0], res["retain"][0])
    for k, a in res["export"][1].items():
        b = res["retain"][1][k]
        scale = float(a.abs().max())
        assert float((a - b).abs().max()) <= 1e-4 * scale + 1e-12, (k, float((a - b).abs().max()), scale)
    # without either switch the backward is refused
    hs = B.HyrfScene(s, mlp_path=B.HYRF_MLP_FMA)
    hs.render(cam)
    with pytest.raises(B.HyrfError) as e:
        hs.backward(g)
    assert e.value.status == B.HYRF_ERR_NOT_READY
    hs.close()


def test_depth_sort_over_a_wide_depth_range(B, ho, synth):
    # csrc/radix.cu sorts the digits of key - bits(z_near) and the host bounds the key bits per frame from max |position|
    # (api.cu): depths within 2^16 : 1 of z_near take three passes, wider ranges a fourth. Both cases, and a scene whose
    # bound changes with a re-upload, against the oracle's per-tile lists bit for bit. The far Gaussians sit on the
    # optical axis region so that they stay in the frustum; the low-pass of D8 keeps them at least a pixel wide.
    rng = np.random.default_rng(5)
    for far, label in ((40.0, "near_only"), (3.0e3, "three_passes"), (2.0e5, "four_passes")):
        s = synth.make_scene(2, n_gaussians=6000, width=200, height=136, n_cameras=2, seed=77)
        cam = s.cameras[0]
        R = cam.R.astype(np.float64)
        eye = -(R.T @ cam.t.astype(np.float64))
        n_far = 400
        z = np.exp(rng.uniform(np.log(5.0), np.log(far), n_far))
        lateral = rng.uniform(-0.2, 0.2, (n_far, 2)) * z[:, None]          # well inside the 60 degree frustum
        p = eye[None, :] + z[:, None] * R[2][None, :] + lateral[:, :1] * R[0][None, :] + lateral[:, 1:] * R[1][None, :]
        s.pos[:, :n_far] = p.T.astype(np.float32)
        s.opacity_logit[:n_far] = 2.0
        st = _run(B, ho, s, exact=True, label=f"wide_depth_{label}")
        assert st[0]["V"] >= n_far // 2


def test_bin_granularity_changes_no_bit(B, ho, synth):
    # hyrf_set_bin_granularity: macro tiles of 2 x 2 .. 16 x 16 tiles (and the per-frame choice) must give the image, the
    # final transmittance and — through the debug export — every per-tile list of the 4 x 4 default, which the other tests
    # compare with the oracle. Large splats over a 3 600-tile frame (the case the coarse settings are chosen for) and
    # the config-3 recipe; then the same against the oracle directly with 8 x 8 macro tiles.
    import torch
    for s in (_adversarial_scene(synth, n=400, W=1280, H=720, seed=41),
              synth.make_scene(3, n_gaussians=100_000, width=1280, height=720, n_cameras=1)):
        cam = s.cameras[0]
        outs = {}
        for shift in (2, 1, 3, 4, 0):
            hs = B.HyrfScene(s, mlp_path=B.HYRF_MLP_FMA)
            hs.set_bin_granularity(shift)
            hs.debug_enable((1 << B.DBG_TILE_LIST) | (1 << B.DBG_TILE_RANGES))
            for _ in range(2):                       # (the per-frame choice looks at the previous frame)
                o = hs.render(cam)
            torch.cuda.synchronize()
            outs[shift] = (o.cpu().numpy().copy(), hs.debug_fetch(B.DBG_FINAL_T).copy(),
                           hs.debug_fetch(B.DBG_TILE_LIST).copy(), hs.debug_fetch(B.DBG_TILE_RANGES).copy())
            hs.close()
        for shift in (1, 3, 4, 0):
            for a, b in zip(outs[2], outs[shift]):
                assert a.shape == b.shape and (a.view(np.uint8) == b.view(np.uint8)).all(), shift
        with pytest.raises(B.HyrfError):
            hs = B.HyrfScene(s); hs.set_bin_granularity(5)
    _run(B, ho, _adversarial_scene(synth, n=400, W=1280, H=720, seed=41), bin_shift=3, label="adversarial_bin8x8")
