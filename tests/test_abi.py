"""CPU-side checks of the boundary: libhyrf.so builds, loads without a GPU and exports every symbol that
include/hyrf.h declares; argument validation that needs no device; multi-rank camera sharding over gloo."""
import ctypes as C
import os
import re
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2509_17083_b200 import build, binding
    build.build()
    return binding.load_library()


def test_every_declared_symbol_is_exported(lib):
    from paper_2509_17083_b200 import binding
    hdr = open(os.path.join(ROOT, "include", "hyrf.h")).read()
    declared = set(re.findall(r"\b(hyrf_[a-z0-9_]+)\s*\(", hdr))
    assert declared == set(binding.EXPORTS), declared ^ set(binding.EXPORTS)
    for name in declared:
        assert hasattr(lib, name), name


def test_struct_layouts_match_header_sizes():
    # sizes computed by the C compiler from the header itself
    from paper_2509_17083_b200 import binding
    src = ('#include "hyrf.h"\n#include <stdio.h>\nint main(){printf("%zu %zu %zu %zu %zu %zu ", '
           'sizeof(hyrf_scene_desc), sizeof(hyrf_params), sizeof(hyrf_camera), sizeof(hyrf_grid_desc), '
           'sizeof(hyrf_mlp_desc), sizeof(hyrf_explicit_rvq));printf("%zu\\n", sizeof(hyrf_grads));return 0;}')
    exe = "/tmp/hyrf_sizes"
    subprocess.run(["gcc", "-x", "c", "-I", os.path.join(ROOT, "include"), "-o", exe, "-"], input=src.encode(),
                   check=True)
    sizes = [int(x) for x in subprocess.run([exe], capture_output=True, check=True).stdout.split()]
    assert sizes == [C.sizeof(binding.SceneDesc), C.sizeof(binding.Params), C.sizeof(binding.CameraC),
                     C.sizeof(binding.GridDesc), C.sizeof(binding.MlpDesc), C.sizeof(binding.ExplicitRvqC),
                     C.sizeof(binding.GradsC)]


def test_argument_validation_without_device(lib, synth):
    from paper_2509_17083_b200 import binding as B
    h = C.c_void_p()
    assert lib.hyrf_create_scene(None, C.byref(h)) == B.HYRF_ERR_INVALID_ARG
    assert b"NULL" in lib.hyrf_last_error()
    s = synth.tiny_scene()
    d = B.make_desc(s, 32, 32)
    d.n_gaussians = 0
    assert lib.hyrf_create_scene(C.byref(d), C.byref(h)) == B.HYRF_ERR_INVALID_ARG
    d = B.make_desc(s, 32, 32)
    d.geo_grid.feats = 4
    assert lib.hyrf_create_scene(C.byref(d), C.byref(h)) == B.HYRF_ERR_UNSUPPORTED
    d = B.make_desc(s, 32, 32)
    d.geo_mlp.hidden = 512
    assert lib.hyrf_create_scene(C.byref(d), C.byref(h)) == B.HYRF_ERR_UNSUPPORTED
    d = B.make_desc(s, 32, 32)
    d.aabb_max[1] = d.aabb_min[1]
    assert lib.hyrf_create_scene(C.byref(d), C.byref(h)) == B.HYRF_ERR_INVALID_ARG
    assert lib.hyrf_render(None, None, 1, 1, None) == B.HYRF_ERR_INVALID_ARG
    assert lib.hyrf_destroy_scene(None) == B.HYRF_ERR_INVALID_ARG
    import torch
    if not torch.cuda.is_available():
        # a valid descriptor on a box without a GPU must fail loudly, never fall back
        d = B.make_desc(s, 32, 32)
        assert lib.hyrf_create_scene(C.byref(d), C.byref(h)) == B.HYRF_ERR_CUDA
        assert not h.value


def test_product_path_never_imports_oracle():
    pkg = os.path.join(ROOT, "paper_2509_17083_b200")
    for dirpath, _, files in os.walk(pkg):
        if os.path.basename(dirpath) in ("build", "__pycache__"):
            continue
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "hyrf_oracle" not in txt and "import oracle" not in txt and "from oracle" not in txt, f


def test_camera_sharding_world2_gloo(tmp_path):
    """Multi-GPU is frame-parallel replicas: cameras dealt round-robin, the only cross-rank step is
    the max-over-ranks of the timed region. Exercised with 2 gloo ranks on CPU."""
    script = tmp_path / "w.py"
    script.write_text(
        "import os, sys, torch, torch.distributed as dist\n"
        f"sys.path.insert(0, {ROOT!r})\n"
        "from paper_2509_17083_b200 import synth\n"
        "import bench\n"
        "dist.init_process_group('gloo')\n"
        "r, w = dist.get_rank(), dist.get_world_size()\n"
        "mine = synth.shard_cameras(20, r, w)\n"
        "allc = [None] * w\n"
        "dist.all_gather_object(allc, mine)\n"
        "flat = sorted(sum(allc, []))\n"
        "assert flat == list(range(20)), flat\n"
        "assert all(len(a) == 10 for a in allc)\n"
        "t = bench.max_over_ranks(1.0 + r)\n"
        "assert t == float(w), t\n"
        "tot = bench.sum_over_ranks(3.0)\n"
        "assert tot == 3.0 * w\n"
        "dist.destroy_process_group()\n")
    env = dict(os.environ, MASTER_ADDR="127.0.0.1", MASTER_PORT="29513")
    r = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2",
                        "--master-addr", "127.0.0.1", "--master-port", "29513", str(script)],
                       capture_output=True, text=True, env=env, timeout=300)
    assert r.returncode == 0, r.stdout + r.stderr


def test_screen_strips_world2_gloo(tmp_path):
    """NEXT-4: screen strips. Each of 2 gloo ranks holds only ITS strip of rows of the oracle's image
    (what hyrf_set_strip leaves in out_rgb on a device); after bench.gather_strips every rank must hold the whole image
    bit for bit. Also the partition itself: strips tile the image, are multiples of 64 rows, the last takes the rest."""
    script = tmp_path / "s.py"
    script.write_text(
        "import os, sys, numpy as np, torch, torch.distributed as dist\n"
        f"sys.path.insert(0, {ROOT!r})\n"
        "from paper_2509_17083_b200 import synth\n"
        "from oracle import hyrf_oracle as ho\n"
        "import bench\n"
        "dist.init_process_group('gloo')\n"
        "r, w = dist.get_rank(), dist.get_world_size()\n"
        "for H in (720, 64, 100, 2160, 1):\n"
        "    for world in (1, 2, 3, 8):\n"
        "        rows = [synth.strip_rows(H, k, world) for k in range(world)]\n"
        "        assert rows[0][0] == 0 and rows[-1][1] == H and all(a[1] == b[0] for a, b in zip(rows, rows[1:])), rows\n"
        "        assert all(a % 64 == 0 for a, _ in rows if a < H)\n"
        "s = synth.make_scene(3, n_gaussians=3000, width=96, height=200, n_cameras=1)\n"
        "img = torch.from_numpy(ho.render(ho.OracleScene(s), s.cameras[0])['out'].copy())\n"
        "H = img.shape[0]\n"
        "y0, y1 = synth.strip_rows(H, r, w)\n"
        "assert (y0, y1) == ((0, 128), (128, 200))[r]\n"
        "mine = torch.full_like(img, float('nan'))\n"
        "mine[y0:y1] = img[y0:y1]\n"
        "got = bench.gather_strips(mine, H, r, w)\n"
        "assert got.shape == img.shape and torch.equal(got.view(torch.int32), img.view(torch.int32))\n"
        "dist.destroy_process_group()\n")
    env = dict(os.environ, MASTER_ADDR="127.0.0.1", MASTER_PORT="29514")
    r = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2",
                        "--master-addr", "127.0.0.1", "--master-port", "29514", str(script)],
                       capture_output=True, text=True, env=env, timeout=300)
    assert r.returncode == 0, r.stdout + r.stderr


def test_explicit_rvq_argument_validation_without_device(lib):
    from paper_2509_17083_b200 import binding as B
    q = B.ExplicitRvqC()
    assert lib.hyrf_upload_explicit_rvq(None, C.byref(q)) == B.HYRF_ERR_INVALID_ARG
    assert lib.hyrf_upload_explicit_rvq(None, None) == B.HYRF_ERR_INVALID_ARG
    ms = C.c_float(0)
    assert lib.hyrf_last_decode_time(None, C.byref(ms)) == B.HYRF_ERR_INVALID_ARG
