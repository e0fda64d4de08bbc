"""bench.py — frames/s and visible Gaussians/s of hyrf_render on one B200 (N>1: frame-parallel replicas).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 3] [--impl ours|reference]

A step = one pass of the whole hot path (S1..S6) for one camera of the workload. Default workload: BASELINE.json
config 3 (1M Gaussians in 64 clusters + far shell, fp16 grids/MLPs, 1280x720, 20 cameras on a circle) — the
config the north_star target is stated on. Inputs are synthetic (paper_2509_17083_b200/synth.py).
`value` is timed with CUDA events on the stream the kernels run on, scene resident in HBM, L2 flushed between
steps; `e2e` goes through hyrf_render_host (camera from host memory, image copied back to pinned host memory).
`--impl reference` times the CPU oracle (oracle/) on the host cores instead.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "frames_per_s"
UNIT = "frames/s"


def _dist():
    import torch.distributed as dist
    return dist if (dist.is_available() and dist.is_initialized()) else None


def max_over_ranks(x: float) -> float:
    d = _dist()
    if d is None:
        return float(x)
    import torch
    dev = "cuda" if d.get_backend() == "nccl" else "cpu"
    t = torch.tensor([float(x)], dtype=torch.float64, device=dev)
    d.all_reduce(t, op=d.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(x: float) -> float:
    d = _dist()
    if d is None:
        return float(x)
    import torch
    dev = "cuda" if d.get_backend() == "nccl" else "cpu"
    t = torch.tensor([float(x)], dtype=torch.float64, device=dev)
    d.all_reduce(t, op=d.ReduceOp.SUM)
    return float(t.item())


def gather_strips(img, H: int, rank: int, world: int, align: int = 64):
    """Screen-strip parallelism (hyrf_set_strip): `img` is a (rows >= H, W, 3) tensor whose rows
    synth.strip_rows(H, rank, world) this rank has rendered; ONE all-gather of equal blocks of rows makes every row valid
    on every rank. With NCCL the gather is in place (each rank's block already sits where it belongs in `img`, which
    must then hold world x block rows); otherwise (gloo, CPU tests) through a staging copy. Returns img[:H]."""
    import torch
    d = _dist()
    block = ((H + align - 1) // align + world - 1) // world * align
    if d is None or world == 1:
        return img[:H]
    begin = min(rank * block, H)
    if d.get_backend() == "nccl" and img.shape[0] >= world * block:
        flat = img[:world * block]
        d.all_gather_into_tensor(flat, flat[rank * block:(rank + 1) * block])
        return img[:H]
    send = torch.zeros((block,) + tuple(img.shape[1:]), dtype=img.dtype, device=img.device)
    n = max(min(H, begin + block) - begin, 0)
    if n:
        send[:n] = img[begin:begin + n]
    parts = [torch.empty_like(send) for _ in range(world)]
    d.all_gather(parts, send)
    full = torch.cat(parts, 0)
    img[:H] = full[:H]
    return img[:H]


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region (B200_PROFILING.md recipe)."""

    def __init__(self, index: int = 0):
        self.index = index
        self.proc = None
        self.lines = []

    def start(self):
        q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
             "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
             "clocks_event_reasons.sw_power_cap")
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={q}", "--format=csv,noheader,nounits",
                                          "-i", str(self.index), "-lms", "100"], stdout=subprocess.PIPE, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, mx, reasons = [], None, set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 8:
                continue
            try:
                sm.append(float(f[0]))
                mx = float(f[1])
            except ValueError:
                continue
            for n, v in zip(names, f[4:8]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": mx, "reasons": sorted(reasons),
                "samples": len(sm)}


def workload(cfg: int, args):
    from paper_2509_17083_b200 import synth
    kw = {}
    if args.n_gaussians:
        kw["n_gaussians"] = args.n_gaussians
    if args.width and args.height:
        kw["width"], kw["height"] = args.width, args.height
    scene = synth.make_scene(cfg, **kw)
    if args.morton_input:
        scene = synth.morton_sorted(scene)
    if args.quant8:
        scene = synth.quantize8(scene)
    if args.rvq:
        scene = synth.compress_explicit(scene, lloyd_iters=1)
    cam = scene.cameras[0]
    name = (f"BASELINE.json configs[{cfg - 1}]: {scene.n} Gaussians, "
            f"{'8-bit tables + fp16 MLPs (compressed model)' if scene.quant8 else ('fp16' if scene.fp16 else 'fp32') + ' grids/MLPs'}, "
            f"{cam.W}x{cam.H}, {len(scene.cameras)} cameras")
    if args.morton_input:
        name += "; Gaussians stored in Morton order (secondary measurement)"
    if scene.explicit_rvq is not None:
        q = scene.explicit_rvq
        name += f"; explicit part compressed (binary16 positions, R-VQ {q.stages} x {q.codebook_size}), decoded at upload"
    return scene, name


# Algorithmic work per unit. Bytes are ALGORITHMIC: what the stage has to move if
# every operand is read once and every result written once, not what the caches happened to move.
def stage_rooflines(scene, V, D, Dm, n_bg, eval_pairs, peaks):
    esz = 1 if scene.quant8 else (2 if scene.fp16 else 4)
    gathers = (scene.geo_grid.levels + scene.app_grid.levels) * 8
    hbm = peaks["hbm_gbs"]
    # S2+S3+S4a: per visible Gaussian 256 gathers of one (2-feature) entry + 32 B explicit record + 4 B work index in;
    # 48 B record + 4 B depth key + 16 B rectangle + 4 B tiles-touched out (1 KB + 32 B + 44-56 B)
    field_bytes = V * (gathers * 2 * esz + 32 + 4 + 48 + 4 + 16 + 4)
    # S1: 16 B of the Morton record + 4 B id read per stored Gaussian, 1 B visibility written; 4 B per visible x 2 lists
    cull_bytes = scene.n * (16 + 4 + 1 + 1) + V * 8
    # S4b-c: depth sort (4 passes x 16 B per visible) + 20 B read per visible for the pairs + 8 B per binned pair
    # written, 4 + 8 B read by count / scatter, 4 B per list entry written. The binned pairs are MACRO-tile entries (Dm).
    bin_bytes = V * (4 * 16 + 4 + 20) + Dm * (8 + 4 + 8 + 4)
    out = {
        "cull": {"bound": "hbm", "work": cull_bytes, "peak": hbm, "unit": "GB/s"},
        "field": {"bound": "hbm", "work": field_bytes, "peak": hbm, "unit": "GB/s"},
        "bin": {"bound": "hbm", "work": bin_bytes, "peak": hbm, "unit": "GB/s"},
    }
    # S5: plain ALU issue. 20 issue slots per evaluated (pixel, Gaussian) pair (16 fp32 ops + ex2 + 3 predicates,
    # SURVEY §8(d)). Peak: the SUSTAINED issue rate measured by the blend-mix microprobe (profiles/r2_probes.json,
    # `python bench.py --probe`), x 32 lanes; without it, the nominal SMs x 4 schedulers x 32 lanes x SM clock.
    alu_nominal = peaks.get("sm_count", 148) * 4 * 32 * peaks.get("sm_max_mhz", 1965.0) * 1e6 / 1e9     # G lane-slots / s
    probes = load_probes()
    alu_peak, alu_src = alu_nominal, "nominal (SMs x 4 x 32 x clock)"
    if probes:
        mix = [v for k, v in probes["issue_warp_instr_per_s_best"].items() if k.startswith("blend mix")]
        if mix:
            alu_peak, alu_src = 32.0 * mix[0] / 1e9, "measured (blend-mix issue probe, profiles/r2_probes.json)"
    if eval_pairs:
        out["raster"] = {"bound": "alu", "work": eval_pairs * 20, "peak": alu_peak, "unit": "Gslot/s",
                         "peak_source": alu_src, "nominal_peak": alu_nominal}
    if n_bg is not None:
        bgl = scene.bg_grid.levels * 8
        out["background"] = {"bound": "hbm", "work": n_bg * (bgl * 2 * esz + 4 + 4 + 12 + 12), "peak": hbm, "unit": "GB/s"}
    return out


def load_traffic(kernel: str):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of `kernel` and, for the field kernel, its L1TEX global-load
    sector look-ups per visible Gaussian, from the committed ncu --set full capture of this workload
    (profiles/r2b_dram_traffic.csv, made by the commands in profiles/r2b_README.md). (None, None) without a capture."""
    p = os.path.join(ROOT, "profiles", "r2b_dram_traffic.csv")
    if not os.path.exists(p):
        return None, None
    import csv
    with open(p) as f:
        for row in csv.DictReader(f):
            if row["kernel"] == kernel:
                sec = row.get("l1tex_ld_sectors_per_visible") or ""
                return float(row["dram_read_bytes"]) + float(row["dram_write_bytes"]), (float(sec) if sec else None)
    return None, None


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            d = json.load(f)
        d["source"] = "measured"
        return d
    return {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0, "sm_max_mhz": 1965.0,
            "source": "fallback"}


def oracle_frames(scene, cams, max_seconds: float, threads: int = 0):
    """Time the CPU oracle as it stands on `cams` (stops after max_seconds). Returns (frames, seconds, V_total,
    threads, evaluated (pixel, Gaussian) pairs as counted by the oracle)."""
    from oracle import hyrf_oracle as ho
    ho.build()
    if threads:
        ho.set_num_threads(threads)
    osc = ho.OracleScene(scene)
    t0 = time.perf_counter()
    frames, vtot, pairs = 0, 0, 0
    for cam in cams:
        r = ho.render(osc, cam)
        frames += 1
        vtot += len(r["vis_idx"])
        pairs += int(r["n_eval"].sum()) if "n_eval" in r else 0
        if time.perf_counter() - t0 > max_seconds:
            break
    return frames, time.perf_counter() - t0, vtot, ho.num_threads(), pairs


def run_reference(args):
    """--impl reference: the oracle timed on the host cores; each step is one frame (bounded sample)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    scene, name = workload(args.config, args)
    cams = scene.cameras
    steps, warm = args.steps, min(args.warmup, 1)
    seq = [cams[i % len(cams)] for i in range(warm + steps)]
    from oracle import hyrf_oracle as ho
    ho.build()
    if args.cpu_threads:
        ho.set_num_threads(args.cpu_threads)     # 1 = the single-thread baseline of SURVEY §8(d); 0 = every host core
    osc = ho.OracleScene(scene)
    for cam in seq[:warm]:
        ho.render(osc, cam)
    t0 = time.perf_counter()
    done = 0
    for cam in seq[warm:]:
        ho.render(osc, cam)
        done += 1
        if time.perf_counter() - t0 > 150:
            break
    dt = time.perf_counter() - t0
    v = done / dt
    line = {"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": done,
            "warmup": warm, "ms_per_step": 1e3 * dt / done, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": name, "note": "CPU oracle (oracle/hyrf_oracle.c) on host cores, one frame per step"},
            "cpu_baseline": {"value": v, "unit": UNIT, "cores": ho.num_threads(), "kind": "oracle",
                             "sample": f"{done} whole frames of the workload"},
            "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line), flush=True)


def run_probe(args):
    """--probe: the two microprobes of SURVEY.md §8(d) (csrc/probe.cu through hyrf_probe_gather / hyrf_probe_issue):
    the scattered-sector look-up ceiling of an L2-resident table and the sustained issue rate of fp32 code. One JSON
    line; the copy kept under profiles/ is what `roofline.l1tex_gather` and the raster `alu` peak refer to."""
    import torch
    from paper_2509_17083_b200 import binding as B
    dev = 0
    torch.cuda.set_device(dev)
    props = torch.cuda.get_device_properties(dev)
    sms = props.multi_processor_count
    sampler = ClockSampler(dev)
    sampler.start()
    gather = []
    for table_mb in (32, 64):
        for eb in (4, 8):
            for ctas in (1, 2, 4, 8):
                lk, sec, ms = B.probe_gather(dev, table_mb << 20, eb, ctas, share=1, line=0, iters=128)
                gather.append({"table_mb": table_mb, "entry_bytes": eb, "ctas_per_sm": ctas, "share": 1, "line": 0,
                               "lookups_per_s": lk, "sectors_per_s": sec, "ms": ms})
    for share, line in ((2, 0), (4, 0), (1, 1), (2, 1)):      # lanes sharing a sector / sectors sharing a line
        for ctas in (2, 4):
            lk, sec, ms = B.probe_gather(dev, 64 << 20, 8, ctas, share=share, line=line, iters=128)
            gather.append({"table_mb": 64, "entry_bytes": 8, "ctas_per_sm": ctas, "share": share, "line": line,
                           "lookups_per_s": lk, "sectors_per_s": sec, "ms": ms})
    issue = []
    for kind, name in ((0, "ffma"), (3, "ffma2 (fma.rn.f32x2: two fma per lane and issue slot)"), (1, "ffma+alu"),
                       (2, "blend mix (1 MUFU.EX2 per 26.75 instructions)")):
        for ctas in (1, 2, 4, 8):
            wi, ms = B.probe_issue(dev, kind, ctas, iters=8192)
            issue.append({"kind": name, "ctas_per_sm": ctas, "warp_instr_per_s": wi, "lane_slots_per_s": 32.0 * wi, "ms": ms})
    clocks = sampler.stop()
    mhz = clocks.get("sm_mhz") or load_peaks().get("sm_max_mhz", 1965.0)
    best_sec = max(g["sectors_per_s"] for g in gather if g["share"] == 1 and g["line"] == 0)
    best_issue = {k: max(i["warp_instr_per_s"] for i in issue if i["kind"] == k) for k in {i["kind"] for i in issue}}
    line = {"probe": "SURVEY.md 8(d) microprobes", "gpu": props.name, "sms": sms, "clocks": clocks,
            "gather_sectors_per_s_best": best_sec, "gather_sectors_per_clk_per_sm": best_sec / (sms * mhz * 1e6),
            "issue_warp_instr_per_s_best": best_issue,
            "issue_per_clk_per_sm": {k: v / (sms * mhz * 1e6) for k, v in best_issue.items()},
            "gather": gather, "issue": issue}
    print(json.dumps(line), flush=True)


def load_probes():
    """profiles/r2_probes.json (written by `python bench.py --probe`), or None."""
    p = os.path.join(ROOT, "profiles", "r2_probes.json")
    if not os.path.exists(p):
        return None
    with open(p) as f:
        return json.load(f)


def run_ours(args):
    import numpy as np
    import torch
    from paper_2509_17083_b200 import binding as B
    from paper_2509_17083_b200 import synth

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world > 1:
        import torch.distributed as dist
        torch.cuda.set_device(local)
        dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local}"))
    dev = local if world > 1 else 0
    torch.cuda.set_device(dev)
    peaks = load_peaks()

    scene, name = workload(args.config, args)
    cams_all = scene.cameras
    strips = args.parallel == "strips" and world > 1
    if strips:
        mine = list(range(len(cams_all)))                   # screen strips: every rank works on every frame
    else:
        mine = synth.shard_cameras(len(cams_all), rank, world) or [rank % len(cams_all)]
    cams = [cams_all[i] for i in mine]                      # frame-parallel replicas: no data-path collective
    path = {"auto": B.HYRF_MLP_AUTO, "fma": B.HYRF_MLP_FMA, "mma": B.HYRF_MLP_MMA, "hmma": B.HYRF_MLP_HMMA, "ws": B.HYRF_MLP_WS}[args.mlp]
    hs = B.HyrfScene(scene, device=dev, mlp_path=path)
    hs.set_ablation(args.ablation)
    hs.set_raster_mode({"auto": 0, "tile": 1, "warp": 2, "pair": 3, "pairall": 4}[args.raster])
    upload = None
    if scene.explicit_rvq is not None:
        # the decode is an upload-time kernel (csrc/decode.cu), not part of a frame: timed on its own, device sources,
        # L2 flushed before each repetition; algorithmic bytes per Gaussian = 6 (binary16 position) + 2 S (codes) + 32 out
        q = scene.explicit_rvq
        flush0 = torch.empty(256 << 20, dtype=torch.uint8, device=f"cuda:{dev}")
        ts = []
        for _ in range(7):
            flush0.fill_(1)
            hs.upload_explicit_rvq(q)
            ts.append(hs.last_decode_time())
        del flush0
        ms = float(np.median(ts[2:]))
        work = scene.n * (6 + 2 * q.stages + 32)
        plain = scene.n * 32
        upload = {"kernel": "explicit_decode_kernel", "decode_ms": ms, "bound": "hbm", "achieved": work / (ms * 1e-3) / 1e9,
                  "peak": peaks["hbm_gbs"], "unit": "GB/s", "frac": work / (ms * 1e-3) / 1e9 / peaks["hbm_gbs"],
                  "explicit_bytes_compressed": q.nbytes(), "explicit_bytes_fp32": plain}
    W, H = cams[0].W, cams[0].H
    out = torch.empty((H, W, 3), dtype=torch.float32, device=f"cuda:{dev}")
    if strips:
        # S1-S4a replicated, S4b-S6 on this rank's strip of tile rows, then one all-gather of H/G x W x 3 floats; the
        # image buffer holds G equal blocks of rows so that the gather is in place
        y0, y1 = synth.strip_rows(H, rank, world)
        block = ((H + 63) // 64 + world - 1) // world * 64
        out = torch.empty((world * block, W, 3), dtype=torch.float32, device=f"cuda:{dev}")
        hs.set_strip(y0, y1) if y1 > y0 else hs.set_strip(0, 16)     # (a rank beyond the image still joins the collective)
    cstructs = [B.camera_struct(c) for c in cams]
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=f"cuda:{dev}")      # > 126 MB L2
    stream = torch.cuda.current_stream(dev)
    K, Wm = args.steps, max(args.warmup, 3)

    def step(i):
        hs.render_struct(cstructs[i % len(cstructs)], W, H, out.data_ptr())
        if strips:
            gather_strips(out, H, rank, world)

    for i in range(Wm):
        step(i)
    torch.cuda.synchronize()

    # --- timed region: K steps, CUDA events on the launching stream, L2 flushed between steps -----------------
    # Each step is bracketed by its own event pair (the flush sits outside the bracket); the library's per-stage
    # events (cudaEventRecord on the same stream, between the kernels) are read after every step, so the kernel
    # durations behind `roofline` come from this very region.
    sampler = ClockSampler(dev)
    sampler.start()
    hs.set_timing(True)
    if world > 1:
        torch.distributed.barrier()
    torch.cuda.synchronize()
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(K)]
    launches = 0
    stage, Vs, Ds, Dms = [], [], [], []
    for i in range(K):
        flush.fill_(i & 0xFF)
        evs[i][0].record(stream)
        step(Wm + i)
        evs[i][1].record(stream)
        launches += hs.last_launch_count()
        stage.append(hs.stage_times())                 # synchronises the stream; outside the bracket
        c = hs.debug_fetch(B.DBG_COUNTERS)
        Vs.append(int(c[1]))
        Ds.append(int(c[2]))
        Dms.append(int(c[4]))
    torch.cuda.synchronize()
    if world > 1:
        torch.distributed.barrier()
    clocks = sampler.stop()
    hs.set_timing(False)
    t_ms = sum(a.elapsed_time(b) for a, b in evs)
    t_max = max_over_ranks(t_ms)
    frames_total = float(K) if strips else sum_over_ranks(K)      # strips: the ranks share every frame (strong scaling)
    value = frames_total / (t_max * 1e-3)
    import numpy as np
    stage_ms = np.mean(np.array(stage), axis=0)
    Vm, Dm, Dmm = float(np.mean(Vs)), float(np.mean(Ds)), float(np.mean(Dms))
    vis_per_s = (Vm * K if strips else sum_over_ranks(Vm * K)) / (t_max * 1e-3)
    n_bg = float((hs.debug_fetch(B.DBG_FINAL_T) > scene.tau_T).sum())        # last frame's S6 work list length

    # --- warm-L2 figure (no flush), for context ---------------------------------------------------------------
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for i in range(K):
        step(i)
    e1.record(stream)
    torch.cuda.synchronize()
    warm_ms = e0.elapsed_time(e1) / K
    # the same stream of frames pipelined (hyrf_set_pipelining: frame k+1's cull and depth sort beside frame k's
    # rasterizer, field kernel on every SM); context for e2e, which adds the device->host copies
    hs.set_pipelining(True)
    for i in range(3):
        step(i)
    torch.cuda.synchronize()
    e0.record(stream)
    for i in range(K):
        step(i)
    e1.record(stream)
    torch.cuda.synchronize()
    pipe_ms = e0.elapsed_time(e1) / K
    hs.set_pipelining(False)

    # --- the same frames with the depth sort serialised (hyrf_set_sort_overlap(0)): every kernel alone on the GPU, the
    # stage times per-kernel profiling sees; reported beside the timed (overlapped) ones, never instead of them -------
    hs.set_sort_overlap(False)
    hs.set_timing(True)
    Ks = min(K, 10)
    step(0)
    torch.cuda.synchronize()
    stage_serial = []
    for i in range(Ks):
        flush.fill_(i & 0xFF)
        step(Wm + i)
        stage_serial.append(hs.stage_times())
    torch.cuda.synchronize()
    hs.set_timing(False)
    hs.set_sort_overlap(True)
    stage_serial_ms = np.mean(np.array(stage_serial), axis=0)
    step(0)
    torch.cuda.synchronize()

    # --- end to end through the public host API: camera from host memory, image back to pinned host memory -------
    # hyrf_render_host_async is the call a user rendering a stream of frames makes: the 11 MB device->host copy of
    # frame k overlaps the render of frame k+1 (two pinned host images, alternating); the clock stops after
    # hyrf_host_sync, when every image is in host memory. e2e_sync is the one-frame-at-a-time hyrf_render_host.
    host_imgs = [torch.empty((H, W, 3), dtype=torch.float32).pin_memory() for _ in range(2)]
    if strips:
        # strips: a frame is complete after the all-gather; rank 0 then delivers it to pinned host memory
        e2e_sync = None
        for i in range(2):
            step(i)
        torch.cuda.synchronize()
        torch.distributed.barrier()
        t0 = time.perf_counter()
        for i in range(K):
            step(i)
            if rank == 0:
                host_imgs[i & 1].copy_(out[:H], non_blocking=True)
        torch.cuda.synchronize()
        e2e_s = max_over_ranks(time.perf_counter() - t0)
        e2e = frames_total / e2e_s
    else:
        for i in range(2):
            hs.render_host(cams[i % len(cams)], out=host_imgs[0])
        t0 = time.perf_counter()
        for i in range(K):
            hs.render_host(cams[i % len(cams)], out=host_imgs[0])
        torch.cuda.synchronize()
        e2e_sync = K / (time.perf_counter() - t0)
        for i in range(2):
            hs.render_host_async(cstructs[i % len(cstructs)], W, H, host_imgs[i & 1])
        hs.host_sync()
        if world > 1:
            torch.distributed.barrier()
        t0 = time.perf_counter()
        for i in range(K):
            hs.render_host_async(cstructs[i % len(cstructs)], W, H, host_imgs[i & 1])
        hs.host_sync()
        e2e_s = max_over_ranks(time.perf_counter() - t0)
        e2e = frames_total / e2e_s
    # what the copies alone cost on this box: the same K images device -> pinned host, nothing else
    dimg = torch.empty((H, W, 3), dtype=torch.float32, device=f"cuda:{dev}")
    host_imgs[0].copy_(dimg, non_blocking=True)
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for i in range(K):
        host_imgs[i & 1].copy_(dimg, non_blocking=True)
    torch.cuda.synchronize()
    d2h_gbs = K * W * H * 12 / (time.perf_counter() - t0) / 1e9

    raster_mode_used = hs.last_raster_mode()
    backward = None
    if args.backward and rank == 0:
        # NEXT-3, first piece: hyrf_raster_backward for camera 0's frame (per-tile lists retained), outside the timed
        # frames; CUDA events on the launching stream, L2 flushed before each repetition
        # the forward pass in training mode (hyrf_set_retain_lists: per-tile ranges from a count-only tile-level binning,
        # lists written by the rasterizer up to its early exit), timed like the inference frames beside it
        def frame_ms(reps=8):
            t = []
            for i in range(reps):
                flush.fill_(1)
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record(stream)
                hs.render_struct(cstructs[i % len(cstructs)], W, H, out.data_ptr())
                e1.record(stream)
                torch.cuda.synchronize(dev)
                t.append(e0.elapsed_time(e1))
            return float(np.median(t[2:]))
        fwd_plain = frame_ms()
        hs.set_retain_lists(True)
        fwd_retain = frame_ms()
        hs.render_struct(cstructs[0], W, H, out.data_ptr())
        torch.cuda.synchronize(dev)
        cnt = hs.debug_fetch(B.DBG_COUNTERS)
        g_c = torch.randn((H, W, 3), dtype=torch.float32, device=f"cuda:{dev}")
        g_t = torch.randn((H, W), dtype=torch.float32, device=f"cuda:{dev}")
        ts = []
        for _ in range(8):
            flush.fill_(1)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            hs.raster_backward(g_c, g_t, int(cnt[1]))
            e1.record(stream)
            torch.cuda.synchronize(dev)
            ts.append(e0.elapsed_time(e1))
        backward = {"kernel": "raster_backward_kernel", "ms": float(np.median(ts[2:])), "V": int(cnt[1]), "D": int(cnt[2]),
                    "note": "includes the memset of the [V][9] gradient rows",
                    "forward_ms": fwd_plain, "forward_retain_lists_ms": fwd_retain}
        # the whole training step's backward: Eq. 12 loss + dL/d image, then hyrf_backward (S6 -> S5 ->
        # S4a -> S3 -> S2 to every parameter): a thread per Gaussian, weight gradients on the tensor cores
        target = torch.rand((H, W, 3), dtype=torch.float32, device=f"cuda:{dev}")
        grads = None
        tl, tb = [], []
        for _ in range(6):
            flush.fill_(1)
            e0, e1, e2 = (torch.cuda.Event(enable_timing=True) for _ in range(3))
            e0.record(stream)
            loss, g_img = hs.loss_l1_ssim(out, target, 0.2)
            e1.record(stream)
            grads = hs.backward(g_img, grads)
            e2.record(stream)
            torch.cuda.synchronize(dev)
            tl.append(e0.elapsed_time(e1)); tb.append(e1.elapsed_time(e2))
        backward.update({"loss_l1_ssim_ms": float(np.median(tl[2:])), "whole_backward_ms": float(np.median(tb[2:])),
                         "loss": loss, "whole_backward_note": "hyrf_backward: background, rasterizer, projection, Eq. 7, decoders, "
                         "grid scatter-adds; gradients of all parameters accumulated over the repetitions"})
        # roofline of the whole backward: it is a CUDA-core pass, so the bound is fp32 issue. Useful
        # work = the decoders' multiply-adds per visible Gaussian, three times over (activations recomputed, deltas
        # propagated, weight gradients: one fma per weight each) + the same for the background pixels; peak = the FFMA
        # rate of the issue microprobe (nominal 4 per clock and SM without it)
        nw = lambda m: sum(o * i for o, i in m.layer_shapes())
        fmas = 3.0 * (nw(scene.geo_mlp) + nw(scene.app_mlp)) * int(cnt[1]) + 3.0 * nw(scene.bg_mlp) * float(n_bg)
        pr = load_probes()
        ffma = pr["issue_warp_instr_per_s_best"].get("ffma") if pr else None
        peak_fma = 32.0 * ffma if ffma else 32.0 * 4.0 * torch.cuda.get_device_properties(dev).multi_processor_count * peaks["sm_max_mhz"] * 1e6
        ach = fmas / (backward["whole_backward_ms"] * 1e-3)
        backward["roofline"] = {"bound": "alu", "achieved": ach / 1e12, "peak": peak_fma / 1e12, "unit": "Tfma/s", "frac": ach / peak_fma,
                                "peak_source": "measured (FFMA issue probe, profiles/r2_probes.json)" if ffma else "nominal",
                                "fma_per_visible_gaussian": 3.0 * (nw(scene.geo_mlp) + nw(scene.app_mlp)),
                                "note": "a thread per Gaussian on CUDA cores (recompute, delta propagation), weight gradients by tf32 mma.sync"}
        hs.set_retain_lists(False)

    if rank != 0:
        return
    names = ["cull", "field", "bin", "raster", "background"]
    kernels = {"field": {"hmma": "field_warp_kernel", "mma": "field_mma_pipe_kernel"}.get(args.mlp, "field_ws_kernel") if scene.fp16 and args.mlp != "fma"
               else "field_fma_kernel", "raster": {2: "raster_warp_kernel", 3: "raster_pair_kernel", 4: "raster_pair_kernel"}.get(raster_mode_used, "raster_kernel")}
    eval_pairs = None
    cpu = None
    if world == 1 and not args.no_cpu and args.ablation == 0:
        fr, sec, vtot, thr, pairs = oracle_frames(scene, [cams_all[i] for i in mine], max_seconds=args.cpu_seconds)
        eval_pairs = pairs / fr
        cpu = {"value": fr / sec, "unit": UNIT, "cores": thr, "kind": "oracle",
               "sample": f"{fr} whole frame(s) of the workload ({vtot / fr:.0f} visible Gaussians each)"}
    peaks["sm_count"] = torch.cuda.get_device_properties(dev).multi_processor_count
    probes = load_probes()
    rl = stage_rooflines(scene, Vm, Dm, Dmm, n_bg, eval_pairs, peaks)
    per_stage = {}
    for i, n in enumerate(names):
        if n in rl:
            r = rl[n]
            ach = r["work"] / (stage_ms[i] * 1e-3) / 1e9
            per_stage[n] = {"bound": r["bound"], "achieved": ach, "peak": r["peak"], "unit": r["unit"],
                            "frac": ach / r["peak"], "ms": float(stage_ms[i])}
            if "nominal_peak" in r:
                per_stage[n].update({"peak_source": r["peak_source"], "frac_of_nominal": ach / r["nominal_peak"]})
    # the dominant KERNEL: S2+S3+S4a and S5 are one kernel each; S4b-c is nine short ones
    dom = "field" if stage_ms[1] >= stage_ms[3] else "raster"
    traffic, sec_per_vis = load_traffic(kernels[dom]) if args.config == 3 else (None, None)
    roof = {"kernel": kernels[dom], "stage": dom, "traffic": traffic,
            "peak_source": per_stage.get(dom, {}).get("peak_source") or
                           (peaks["source"] + (" (burst HBM copy)" if per_stage.get(dom, {}).get("bound") == "hbm" else ""))}
    if dom in per_stage:
        roof.update({k: per_stage[dom][k] for k in ("bound", "achieved", "peak", "unit", "frac")})
        roof["launch_ms"] = per_stage[dom]["ms"]
        # the same kernel with the GPU to itself (serialised frame): its own ceiling, without the sort's CTAs beside it
        di = names.index(dom)
        roof["serial_launch_ms"] = float(stage_serial_ms[di])
        roof["serial_frac"] = rl[dom]["work"] / (stage_serial_ms[di] * 1e-3) / 1e9 / rl[dom]["peak"]
    else:
        # the rasterizer's work is counted in evaluated (pixel, Gaussian) pairs, which only the CPU oracle leg counts
        roof.update({"bound": "alu", "achieved": None, "peak": None, "unit": "Gslot/s", "frac": None,
                     "note": "the dominant kernel is the rasterizer; its pair count comes from the cpu_baseline leg (run without --no-cpu / --ablation)"})
    # What actually bounds the field kernel (its tables are L2-resident, DRAM moves a sixth of the algorithmic bytes): the
    # rate at which an SM looks up scattered sectors. Achieved = the kernel's L1TEX global-load sector look-ups (ncu count
    # per visible Gaussian of the committed capture x this run's V) / its launch time; peak = the gather microprobe.
    _, field_sec = load_traffic(kernels["field"]) if args.config == 3 else (None, None)
    if probes and field_sec:
        ach = field_sec * Vm / (stage_ms[1] * 1e-3)
        roof_l1 = {"bound": "l1tex_gather", "kernel": kernels["field"], "achieved": ach / 1e9, "peak": probes["gather_sectors_per_s_best"] / 1e9,
                   "unit": "Gsector/s", "frac": ach / probes["gather_sectors_per_s_best"],
                   "sectors_per_visible_gaussian": field_sec, "peak_source": "measured (gather microprobe, profiles/r2_probes.json)"}
        if dom == "field":
            roof["l1tex_gather"] = roof_l1
        per_stage["field"]["l1tex_gather"] = roof_l1
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": Wm,
            "ms_per_step": t_max / K, "higher_is_better": True, "scaling": "strong" if strips else "weak", "vs_baseline": None,
            "dtype": "f16" if scene.fp16 else "f32", "data": "synthetic",
            "config": {"workload": name, "l2": "flushed between steps (256 MiB write)", "mlp_path": args.mlp, "ablation": args.ablation, "raster": args.raster,
                       "schedule": "one frame at a time; S1 + depth sort on the library's second stream, the sort beside the field kernel (hyrf_set_sort_overlap default); e2e: frames pipelined (hyrf_render_host_async)",
                       "parallelism": (f"screen strips x{world} (S1-S4a replicated, S4b-S6 per strip, one all-gather per frame)" if strips
                                       else f"replicas x{world} (cameras round-robin)")},
            "visible_gaussians_per_s": vis_per_s, "V_mean": Vm, "D_mean": Dm, "Dm_mean": Dmm,
            "stage_ms": {n: float(stage_ms[i]) for i, n in enumerate(names)} | {"frame": float(stage_ms[5])},
            "serial_stage_ms": {n: float(stage_serial_ms[i]) for i, n in enumerate(names)} | {"frame": float(stage_serial_ms[5])},
            "warm_l2_ms_per_step": warm_ms, "pipelined_warm_l2_ms_per_step": pipe_ms,
            "e2e": {"value": e2e, "unit": UNIT, "h2d_bytes_per_step": 64, "d2h_bytes_per_step": W * H * 12,
                    "api": "hyrf_render (strip) + all-gather + copy to pinned host on rank 0" if strips else "hyrf_render_host_async + hyrf_host_sync",
                    "sync_api_value": e2e_sync,
                    "d2h_copy_only_gbs": d2h_gbs, "d2h_copy_only_frames_per_s": d2h_gbs * 1e9 / (W * H * 12)},
            "gpu_launches": launches, "clocks": clocks, "roofline": roof, "stage_rooflines": per_stage}
    if cpu:
        line["cpu_baseline"] = cpu
    if upload:
        line["upload_decode"] = upload
    if backward:
        line["backward"] = backward
    print(json.dumps(line), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--mlp", default="auto", choices=["auto", "fma", "mma", "hmma", "ws"])
    ap.add_argument("--n-gaussians", type=int, default=0)
    ap.add_argument("--width", type=int, default=0)
    ap.add_argument("--height", type=int, default=0)
    ap.add_argument("--ablation", type=int, default=0,
                    help="hyrf_ablation bits (PAPER.md Table 5): 1 no pre-culling, 2 no background, 4 no neural, 8 no explicit")
    ap.add_argument("--quant8", action="store_true",
                    help="compressed model: 8-bit min-max tables decoded in the gather (PAPER.md:229)")
    ap.add_argument("--raster", default="auto", choices=["auto", "tile", "warp", "pair", "pairall"],
                    help="hyrf_set_raster_mode: per-frame choice (default), tile-level lists only, per-warp lists")
    ap.add_argument("--morton-input", action="store_true",
                    help="store the Gaussians in Morton order of their positions (SURVEY 8(d): secondary, labelled measurement)")
    ap.add_argument("--backward", action="store_true",
                    help="also time hyrf_raster_backward (backward of the alpha blend, NEXT-3 first piece) on camera 0's frame")
    ap.add_argument("--rvq", action="store_true",
                    help="compressed explicit Gaussians: binary16 positions + R-VQ codes decoded at upload (PAPER.md:229 (1)-(2))")
    ap.add_argument("--parallel", default="replicas", choices=["replicas", "strips"],
                    help="N > 1: frame-parallel replicas (default, no data-path collective) or screen strips with one "
                         "all-gather per frame (SURVEY 8(e)(2); pays at the 4K / 4M points of config 5)")
    ap.add_argument("--probe", action="store_true",
                    help="run the L2 gather and issue-rate microprobes of SURVEY 8(d) instead of the render benchmark")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--cpu-seconds", type=float, default=15.0)
    ap.add_argument("--cpu-threads", type=int, default=0,
                    help="--impl reference: OpenMP threads of the oracle (0 = all host cores, 1 = single-thread baseline)")
    args = ap.parse_args()
    if args.probe:
        run_probe(args)
    elif args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)
    d = _dist()
    if d is not None:
        d.destroy_process_group()


if __name__ == "__main__":
    main()
