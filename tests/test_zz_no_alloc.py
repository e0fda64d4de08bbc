"""hyrf_loss_l1_ssim_noalloc (include/hyrf.h): the Eq. 12 loss through the entry point that allocates nothing, against
the existing hyrf_loss_l1_ssim on the same inputs. Collected last on purpose (pytest -x)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2509_17083_b200 import binding
    binding.load_library()          # raises if the extension is missing: no silent fallback
    return binding


def _pair(torch, H, W, seed):
    g = torch.Generator(device="cuda").manual_seed(seed)
    target = torch.rand((H, W, 3), generator=g, device="cuda")
    image = (target + 0.2 * torch.randn((H, W, 3), generator=g, device="cuda")).clamp_(0, 1).contiguous()
    return image, target


def test_noalloc_loss_matches_the_scene_path_twice_in_a_row(B, synth):
    import torch
    s = synth.tiny_scene(n=16, W=160, H=96)
    hs = B.HyrfScene(s)
    # two calls in a row on the shared scratch: the second on a smaller image with other contents, so anything the first
    # call left behind (accumulator, maps laid out for another W x H) would show
    for k, (H, W) in enumerate([(96, 160), (37, 45)]):
        image, target = _pair(torch, H, W, seed=100 + k)
        want_L, want_g = hs.loss_l1_ssim(image, target, 0.2)
        g = torch.full_like(image, float("nan"))
        torch.cuda.synchronize()
        before = torch.cuda.memory_allocated()
        got_L = B.loss_l1_ssim_noalloc(image, target, 0.2, g)
        assert torch.cuda.memory_allocated() == before
        # same kernels, same operations: the gradient agrees bit for bit, the loss up to the order of its atomic adds;
        # the tolerances are those of test_backward_against_oracle for the same quantities
        assert abs(got_L - want_L) <= 1e-5 * abs(want_L), (k, got_L, want_L)
        err = (g - want_g).abs().max().item()
        scale = want_g.abs().max().item()
        assert np.isfinite(g.cpu().numpy()).all()
        assert err <= 1e-4 * scale, (k, err, scale)
        # without a gradient buffer only the loss comes back
        assert abs(B.loss_l1_ssim_noalloc(image, target, 0.2) - want_L) <= 1e-5 * abs(want_L)
    hs.close()


def test_noalloc_loss_rejects_what_does_not_fit(B):
    import torch
    z = torch.zeros((1, 1, 3), device="cuda")
    with pytest.raises(B.HyrfError) as e:   # 1025 x 1024 pixels > HYRF_LOSS_NOALLOC_MAX_PIXELS: refused before any launch
        B._check(B.load_library().hyrf_loss_l1_ssim_noalloc(0, None, z.data_ptr(), z.data_ptr(), 1025, 1024, 0.2,
                                                             B.C.byref(B.C.c_double(0)), None))
    assert e.value.status == B.HYRF_ERR_INVALID_ARG and "exceed" in str(e.value)
    image, target = _pair(torch, 1024, 1024, seed=7)   # the largest size that fits runs
    L = B.loss_l1_ssim_noalloc(image, target, 0.2)
    assert 0.0 < L < 1.0
