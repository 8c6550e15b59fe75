#!/usr/bin/env python
"""bench.py — one JSON line for the LEGS hot path on B200 (contract: see DESIGN.md "Measurement").

A step = one pass of the whole hot path over one synthetic view of BASELINE.json configs[2] (1M Gaussians, 1600x1064,
SH degree 3, F = 8 + uncertainty): legs_preprocess -> legs_bin_and_sort -> legs_render_forward -> legs_render_backward
-> legs_decode_semantics (configs[3] decoder 8->64->128, 128x896 codebook, probs + decoded) -> legs_relevancy.
metric = BASELINE.json's (megapixels/s = W*H / time). `value` times the whole step with every input resident in HBM; the
two numbers the metric names, forward (S1-S5) and forward + backward (S1-S7), are the `fwd` and `fwd_bwd` objects, each
with its fraction of the roofline under SURVEY.md 8(d)'s work model and under the model of the algorithm as built;
`e2e` times the same calls with host buffers (pinned) copied in and results copied out inside the timed region.
The FP32-issue and MUFU ex2 peaks that the ALU rooflines divide by are MEASURED in the same run (legs_peak_kernel).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--small]
N > 1: launched under torchrun, one rank per GPU: the by-view split of SURVEY.md 8(e) -- every rank holds a replica of
the Gaussians and renders its own view forward + backward; the step ends with ONE NCCL all-reduce (sum) of the flat
gradient buffer, the only exchange the split has. value = all ranks' pixels / max-over-ranks time ("weak").
--impl reference times the CPU oracle (oracle/) on a bounded pixel sample of the same workload.
"""
from __future__ import annotations

import argparse
import json
import math
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2311_18482_b200 import inputs  # noqa: E402

METRIC = "megapixels/s fwd and fwd+bwd (RGB+semantic) at 1M Gaussians; % of roofline"   # BASELINE.json `metric`
UNIT = "Mpix/s"


def workload(small: bool):
    if small:
        scene = inputs.unbounded_scene(n=100_000, width=640, height=424, focal=460.0)
        name = "configs[2]-shaped, reduced (100k Gaussians, 640x424)"
    else:
        scene = inputs.unbounded_scene()
        name = "configs[2] unbounded scene: 1M Gaussians, 1600x1064, SH3, F=8+u; decode configs[3] (8->64->128, 128x896)"
    return scene, name


def view_for_rank(scene, rank: int):
    """Rank r looks at the scene from the configs[2] camera rotated by r * 45 degrees about the world y axis."""
    cam0 = scene.cameras[0]
    if rank == 0:
        return cam0
    W = cam0.world_to_cam.astype(np.float64).reshape(3, 4)
    c = -W[:, :3].T @ W[:, 3]
    a = rank * math.pi / 4
    R = np.array([[math.cos(a), 0, math.sin(a)], [0, 1, 0], [-math.sin(a), 0, math.cos(a)]])
    return inputs.look_at_camera(R @ c, cam0.width, cam0.height, cam0.fx, cam0.fy, cam0.cx, cam0.cy)


def aggregate(pixels_per_rank: float, seconds_local: float, world: int, reduce_max=None) -> dict:
    """Whole-job throughput: all ranks' pixels / max-over-ranks time (host logic shared with the gloo test)."""
    t = seconds_local if reduce_max is None else reduce_max(seconds_local)
    return dict(seconds=t, mpix_s=pixels_per_rank * world / t / 1e6)


def nccl_init_lines(path, limit: int = 6):
    """The communicator lines of rank 0's NCCL INIT log (rank count, NVLS / P2P transport), for the JSON line."""
    if not path or not os.path.exists(path):
        return None
    keep = [ln.strip()[-200:] for ln in open(path, errors="replace") if ("nranks" in ln or "Init COMPLETE" in ln or "NVLS" in ln)]
    return keep[:limit]


def free_port() -> int:
    import socket
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        return sk.getsockname()[1]


def relaunch_under_torchrun(args, argv) -> int:
    """`python bench.py --gpus N` with no WORLD_SIZE in the environment: start the N ranks ourselves, the way the driver
    does (python -m torch.distributed.run, one process per GPU, rendezvous on 127.0.0.1). stdout is inherited: rank 0's one
    JSON line is the only thing printed."""
    import subprocess
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}", "--master-addr", "127.0.0.1",
           "--master-port", str(free_port()), os.path.abspath(__file__)] + list(argv)
    return subprocess.run(cmd).returncode


def run_dry_host(args):
    """--dry-host: the N > 1 plumbing of run_gpu without a GPU (gloo, CPU tensors): rank environment, one view per rank, the
    asynchronous all-reduce of the flat gradient buffer issued before the (stand-in) decode stage and waited for after it,
    max-over-ranks timing, and rank 0's single JSON line. No kernel runs and the line carries no throughput claim
    ("dry_host": true); tests/test_multirank_host.py drives it through the launcher above."""
    import torch
    import torch.distributed as dist
    from types import SimpleNamespace
    from paper_2311_18482_b200 import binding
    rank, world = int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))
    if world > 1:
        dist.init_process_group("gloo", rank=rank, world_size=world)
    scene = inputs.unbounded_scene(n=64, width=64, height=64, focal=46.0)
    cam = view_for_rank(scene, rank)
    grads = binding.Grads(SimpleNamespace(n=scene.n, sh_stored=16, F=scene.sem_dim), device="cpu")
    t0 = time.perf_counter()
    for k in range(args.steps):
        grads.flat.fill_(float(rank + 1))                              # stands in for S1-S7 of this rank's view
        work = dist.all_reduce(grads.flat, op=dist.ReduceOp.SUM, async_op=True) if world > 1 else None
        _ = torch.ones(256, 256) @ torch.ones(256, 256)                # stands in for decode + relevancy
        if work is not None:
            work.wait()
    t_local = time.perf_counter() - t0

    def reduce_max(t):
        tt = torch.tensor([t], dtype=torch.float64)
        dist.all_reduce(tt, op=dist.ReduceOp.MAX)
        return float(tt.item())

    agg = aggregate(cam.width * cam.height * args.steps, t_local, world, reduce_max if world > 1 else None)
    want = float(sum(range(1, world + 1)))
    ok = bool((grads.flat == want).all().item())
    views = [None] * world
    if world > 1:
        dist.all_gather_object(views, [float(v) for v in cam.world_to_cam])
        dist.barrier()
        dist.destroy_process_group()
    else:
        views = [[float(v) for v in cam.world_to_cam]]
    if rank == 0:
        print(json.dumps(dict(metric=METRIC, value=None, unit=UNIT, n_gpus=world, steps=args.steps, warmup=args.warmup, dry_host=True,
                              scaling="weak", seconds_max_over_ranks=agg["seconds"], grads_allreduce_ok=ok,
                              distinct_views=len({tuple(v) for v in views}),
                              config=dict(workload="dry host run: no kernels, plumbing only", parallelism=f"by view: {world} replicas"))))


class ClockSampler:
    """Samples nvidia-smi clocks and throttle reasons during the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.samples, self.proc = [], None
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(index), f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", "25"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.samples.append((time.monotonic(), line.strip()))

    def wait_first(self, timeout=5.0):
        """nvidia-smi takes a moment to start: block until its first line arrives (before the timed region)."""
        t0 = time.monotonic()
        while self.proc and not self.samples and time.monotonic() - t0 < timeout:
            time.sleep(0.01)

    def stop(self, t_begin=None, t_end=None) -> dict:
        """Summary of the samples taken inside [t_begin, t_end] (host monotonic clock around the timed region)."""
        if not self.proc:
            return dict(sm_mhz=None, sm_max_mhz=None, reasons=["nvidia-smi unavailable"])
        self.proc.terminate()
        inside = [s for (t, s) in self.samples if (t_begin is None or t >= t_begin) and (t_end is None or t <= t_end + 0.03)]
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for s in inside:
            f = [x.strip() for x in s.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1]))
            except ValueError:
                continue
            for n, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return dict(sm_mhz=float(np.median(sm)) if sm else None, sm_max_mhz=max(mx) if mx else None,
                    reasons=sorted(reasons), samples=len(sm))


def peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        p = json.load(open(path))
        return dict(hbm_gbs=p["hbm_gbs"], bf16=p["bf16_tflops"], bf16_sustained=p.get("bf16_tflops_sustained"), source="measured")
    return dict(hbm_gbs=6650.0, bf16=1590.0, bf16_sustained=1400.0, source="fallback")


# ---------------------------------------------------------------------------------------------------------
# reference arm / cpu_baseline: the oracle on a bounded pixel sample

def oracle_sample_throughput(scene, cam, n_sample: int, seed: int = 0) -> dict:
    from oracle import legs_oracle as O
    O.build()
    P = cam.width * cam.height
    rng = np.random.Generator(np.random.PCG64(seed))
    pix = np.sort(rng.choice(P, size=min(n_sample, P), replace=False)).astype(np.int64)
    CH = inputs.channels(scene.sem_dim)
    G = np.zeros((pix.shape[0], CH))
    G[:, 0:3] = rng.standard_normal((pix.shape[0], 3))
    G[:, 4:5 + scene.sem_dim] = rng.standard_normal((pix.shape[0], scene.sem_dim + 1))
    di = inputs.decode_inputs(P=8, seed=1)
    f32 = inputs.bf16_bits_to_f32
    t0 = time.perf_counter()
    proj = O.project(scene, cam, 0)
    O.tile_lists(proj, cam)
    t_fixed_fwd = time.perf_counter() - t0
    t0 = time.perf_counter()
    fw = O.composite_forward(proj, scene.sem, scene.unc, cam, pix)
    g2 = O.composite_backward(proj, scene.sem, scene.unc, cam, G, pix)
    x = f32(inputs.to_bf16_bits(fw["out"][:, 4:4 + scene.sem_dim].astype(np.float32)))
    O.decode(x, [f32(w) for w in di.weights], di.biases, f32(di.codebook), di.d_clip, f32(di.queries))
    t_pix = time.perf_counter() - t0
    t0 = time.perf_counter()
    O.project_backward(scene, cam, g2, 0)
    t_fixed_bwd = time.perf_counter() - t0
    t_frame = t_fixed_fwd + t_fixed_bwd + t_pix * (P / pix.shape[0])
    cores = len(os.sched_getaffinity(0)) if hasattr(os, "sched_getaffinity") else os.cpu_count()
    return dict(value=P / t_frame / 1e6, unit=UNIT, cores=cores, kind="oracle",
                sample=f"{pix.shape[0]} random pixels of the {cam.width}x{cam.height} view: fwd+bwd compositing and decode timed "
                       f"({t_pix:.2f} s) and scaled to the frame, plus whole-scene projection, tile lists and projection "
                       f"backward ({t_fixed_fwd + t_fixed_bwd:.2f} s)",
                seconds_measured=t_fixed_fwd + t_fixed_bwd + t_pix, ms_per_frame_estimate=t_frame * 1e3)


def oracle_small_configs() -> dict:
    """SURVEY.md 8(d) "Timing": the oracle on configs[0] whole (forward + backward), all cores and single-threaded."""
    import ctypes
    from oracle import legs_oracle as O
    O.build()
    scene = inputs.tiny_scene()
    cam = scene.cameras[0]
    up = inputs.upstream_gradient(scene, 0).reshape(-1, inputs.channels(scene.sem_dim))
    out = {}
    try:
        gomp = ctypes.CDLL("libgomp.so.1")
        ncores = len(os.sched_getaffinity(0))
    except OSError:
        gomp, ncores = None, 1
    for label, threads in (("all_cores", ncores), ("single_thread", 1)):
        if gomp is not None:
            gomp.omp_set_num_threads(threads)
        t0 = time.perf_counter()
        O.render_forward(scene, cam)
        t1 = time.perf_counter()
        O.render_backward(scene, cam, up)
        t2 = time.perf_counter()
        P = cam.width * cam.height
        out[label] = dict(threads=threads, fwd_mpix_s=round(P / (t1 - t0) / 1e6, 4), fwd_bwd_mpix_s=round(P / (t2 - t0) / 1e6, 4))
    if gomp is not None:
        gomp.omp_set_num_threads(ncores)
    return out


def oracle_configs1_whole_frame() -> dict:
    """SURVEY.md 8(d) "Timing": the oracle on ONE WHOLE frame of configs[1] (100k Gaussians, 800x800), forward and forward
    + backward, all cores: 8.7 s + 9.0 s on the 16 host cores of the B200 box (--no-oracle-configs1 skips it)."""
    from oracle import legs_oracle as O
    O.build()
    scene = inputs.object_scene()
    cam = scene.cameras[0]
    up = inputs.upstream_gradient(scene, 0).reshape(-1, inputs.channels(scene.sem_dim))
    P = cam.width * cam.height
    t0 = time.perf_counter()
    O.render_forward(scene, cam)
    t1 = time.perf_counter()
    O.render_backward(scene, cam, up)      # (runs its own forward pass first)
    t2 = time.perf_counter()
    cores = len(os.sched_getaffinity(0)) if hasattr(os, "sched_getaffinity") else os.cpu_count()
    return dict(threads=cores, fwd_s=round(t1 - t0, 2), fwd_mpix_s=round(P / (t1 - t0) / 1e6, 5),
                fwd_bwd_s=round(t2 - t1, 2), fwd_bwd_mpix_s=round(P / (t2 - t1) / 1e6, 5))


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    scene, name = workload(args.small)
    cam = scene.cameras[0]
    vals = []
    res = None
    for i in range(args.warmup + args.steps):
        res = oracle_sample_throughput(scene, cam, args.ref_sample, seed=i)
        if i >= args.warmup:
            vals.append(res)
    v = float(np.mean([r["value"] for r in vals]))
    ms = float(np.mean([r["ms_per_frame_estimate"] for r in vals]))
    line = dict(impl="reference", metric=METRIC, value=v, unit=UNIT, n_gpus=args.gpus, steps=args.steps, warmup=args.warmup,
                ms_per_step=ms, higher_is_better=True, scaling="weak", vs_baseline=None, dtype="f64", data="synthetic",
                config=dict(workload=name, note="CPU oracle, each step a bounded pixel sample scaled to the frame"),
                cpu_baseline=dict(value=v, unit=UNIT, cores=res["cores"], kind="oracle", sample=res["sample"]),
                e2e=dict(value=v, unit=UNIT, h2d_bytes_per_step=0, d2h_bytes_per_step=0))
    print(json.dumps(line))


# ---------------------------------------------------------------------------------------------------------
# GPU arm

def measure_alu_peaks(legs, ctx, torch) -> dict:
    """FP32-issue (FFMA chains) and MUFU ex2 rates of this GPU, measured now.
    Best of 5 launches of ~2.5 ms each, CUDA events on the launching stream."""
    sink = torch.zeros(ctx.num_sms * 8 * 256, dtype=torch.float32, device=ctx.device)
    out = {}
    for kind, name, iters in ((0, "ffma_t_lane_instr_s", 10000), (1, "ex2_t_s", 1200), (2, "ffma2_t_lane_instr_s", 5000)):
        best = 0.0
        for _ in range(6):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            ops = legs.legs_peak_kernel(ctx, kind, iters, sink)
            e1.record()
            torch.cuda.synchronize()
            best = max(best, ops / (e0.elapsed_time(e1) * 1e-3) / 1e12)
        out[name] = round(best, 3)
    return out


NCU_SUMMARY = os.path.join("profiles", "r03_ncu_full_summary.csv")


def ncu_committed(kernel_regex: str):
    """One launch of the named kernel as the committed `ncu --set full` capture saw it (NOT measured in this run; the file
    is named in the returned `source`, so a stale capture is visible): dram__bytes_read.sum + dram__bytes_write.sum,
    smsp__issue_active and smsp__inst_executed.sum (warp instructions). None if the file or the kernel is not there."""
    import csv
    import re
    path = os.path.join(ROOT, NCU_SUMMARY)
    if not os.path.exists(path):
        return None
    with open(path) as f:
        rows = list(csv.reader(f))
    if not rows:
        return None
    head = rows[0]
    def col(prefix):
        for i, h in enumerate(head):
            if h.startswith(prefix):
                return i, h
        return None, None
    ir, hr = col("dram__bytes_read.sum")
    iw, hw = col("dram__bytes_write.sum")
    ii, _ = col("smsp__issue_active")
    ix, _ = col("smsp__inst_executed.sum")
    if ir is None or iw is None:
        return None
    unit = lambda h: {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9}.get(h[h.index("[") + 1:h.index("]")], 1.0)
    for r in rows[1:]:
        if r and re.search(kernel_regex, r[0]):
            return dict(traffic=int(float(r[ir]) * unit(hr) + float(r[iw]) * unit(hw)),
                        issue_active_pct=None if ii is None else round(float(r[ii]), 1),
                        warp_instructions=None if ix is None else int(float(r[ix])),
                        source=NCU_SUMMARY + " (committed ncu --set full capture of this kernel, see profiles/r03_profiles.md; not measured in this run)")
    return None


def time_config(legs, ctx, torch, scene, label: str, flush, alu_peak: float, hbm_gbs: float, step_views: int = 0) -> dict:
    """One view of another BASELINE.json config through S1-S7 (VERDICT r2 missing 2: configs[1] and configs[4], whose
    regime differs in kind from configs[2]'s): per-stage ms over 10 flushed runs after 3 warm-ups, fwd / fwd+bwd ms and
    Mpix/s, and each stage's fraction under the model of the algorithm as built (same formulas as the headline config).
    step_views > 0 also times the config's whole step: that many views rendered forward + backward into one accumulated
    gradient set, each followed by the configs[3]-shaped decode (in_dim = F) and the relevancy map."""
    dev = ctx.device
    g = legs.Gaussians.from_scene(scene, dev)
    cams = scene.cameras[:max(1, step_views)]
    W, H, F = cams[0].width, cams[0].height, scene.sem_dim
    P = W * H
    upstream = torch.from_numpy(inputs.upstream_gradient(scene, 0)).to(dev)
    Ds = []
    for c in cams:
        probe = legs.Renderer(ctx, g, c, capacity=16)
        legs.legs_preprocess(ctx, g, probe.cam, probe.frame)
        Ds.append(legs.legs_read_num_instances(ctx, probe.frame))
        del probe
    r = legs.Renderer(ctx, g, cams[0], capacity=int(max(Ds) * 1.02) + 1024, want_keys=False, want_bf16=True)
    r.bwd_ws = torch.empty(legs.legs_backward_workspace_bytes(g.n, F), dtype=torch.uint8, device=dev)
    order = torch.empty(r.ntiles, dtype=torch.int32, device=dev)   # heavy tiles first (legs_tile_order, timed inside render_forward)
    grads = legs.Grads(g, dev)
    names = ["preprocess", "bin_and_sort", "render_forward", "render_backward"]

    def one(ev=None, flags=0):
        mark = (lambda i: ev[i].record()) if ev is not None else (lambda i: None)
        mark(0)
        legs.legs_preprocess(ctx, g, r.cam, r.frame); mark(1)
        legs.legs_bin_and_sort(ctx, r.frame, r.cam, g.n, r.capacity, None, r.vals_sorted, r.ranges, r.sort_ws); mark(2)
        legs.legs_tile_order(ctx, r.ranges, order); legs.legs_render_forward(ctx, g, r.cam, r.frame, r.vals_sorted, r.ranges, r.out, r.n_contrib, r.sem_bf16, r.block_masks, order); mark(3)
        legs.legs_render_backward(ctx, g, r.cam, r.frame, r.vals_sorted, r.ranges, r.out, r.n_contrib, upstream, flags, grads,
                                  r.bwd_ws, r.block_masks, order); mark(4)

    ms, s6 = [], []
    for k in range(3 + 10):
        flush.fill_(k)
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(7)]
        one(ev)
        flush.fill_(k + 1)
        ev[5].record()
        legs.legs_render_backward(ctx, g, r.cam, r.frame, r.vals_sorted, r.ranges, r.out, r.n_contrib, upstream,
                                  legs.LEGS_BWD_COMPOSITE_ONLY, grads, r.bwd_ws, r.block_masks, order)
        ev[6].record()
        torch.cuda.synchronize()
        if k >= 3:
            ms.append([ev[i].elapsed_time(ev[i + 1]) for i in range(4)])
            s6.append(ev[5].elapsed_time(ev[6]))
    ms, s6 = np.array(ms).mean(0), float(np.mean(s6))
    counters = torch.zeros(4, dtype=torch.int64, device=dev)
    legs.legs_render_forward_stats(ctx, g, r.cam, r.frame, r.vals_sorted, r.ranges, r.out, r.n_contrib, counters)
    torch.cuda.synchronize()
    P_ek, P_b, I_f, P_e = [int(x) for x in counters.cpu().numpy()]
    n, D = g.n, Ds[0]
    n_vis = int((r.frame.tiles_touched > 0).sum().item())
    rect = r.frame.rect.view(-1, 4)
    n_rows = int(((rect[:, 3] - rect[:, 1]) * (r.frame.tiles_touched > 0)).sum().item())
    ntiles = math.ceil(W / 16) * math.ceil(H / 16)
    RSb = 4 * legs.record_stride(F)
    work = {"preprocess": ("hbm", n * (12 + 65) + n_vis * (12 + 16 + 4 + 192 + 4 * F + 4 + RSb)),
            "bin_and_sort": ("hbm", n * (4 + 4 * 16 + 2 * 20) + n_rows * (8 + 8 + 8) + D * 4 + ntiles * 8),
            "render_forward": ("alu", 12 * P_ek + (4 + 3 + F + 2) * P_b),
            "render_backward_s6": ("alu", 12 * P_ek + (75 + 20) * P_b),
            "project_backward_s7": ("hbm", n_vis * (240 + 4 * (10 + F)) + n_vis * (4 * (3 + 3 + 4 + 1 + 48 + F + 1 + 2)))}
    t_of = {"preprocess": ms[0], "bin_and_sort": ms[1], "render_forward": ms[2], "render_backward_s6": s6,
            "project_backward_s7": max(ms[3] - s6, 1e-6)}
    stages = {}
    for nm, (bound, w) in work.items():
        roof_ms = w / (hbm_gbs * 1e9 if bound == "hbm" else alu_peak * 1e12) * 1e3
        stages[nm] = dict(ms=round(float(t_of[nm]), 4), bound=bound, roofline_ms=round(roof_ms, 4), frac_built=round(roof_ms / float(t_of[nm]), 4))
    fwd_ms, fb_ms = float(ms[:3].sum()), float(ms.sum())
    roof_f = sum(stages[k]["roofline_ms"] for k in ("preprocess", "bin_and_sort", "render_forward"))
    roof_fb = roof_f + stages["render_backward_s6"]["roofline_ms"] + stages["project_backward_s7"]["roofline_ms"]
    out = dict(workload=label, n=int(n), width=W, height=H, sem_dim=F, D=int(D), n_visible=n_vis,
               examined_pairs_after_block_culling=P_ek, examined_pairs_plain_walk=P_e, blended_pairs=P_b,
               blended_over_examined=round(P_b / max(P_ek, 1), 4),
               fwd=dict(ms=round(fwd_ms, 4), mpix_s=round(P / fwd_ms / 1e3, 1), frac_built=round(roof_f / fwd_ms, 4)),
               fwd_bwd=dict(ms=round(fb_ms, 4), mpix_s=round(P / fb_ms / 1e3, 1), frac_built=round(roof_fb / fb_ms, 4)),
               stages=stages)
    if step_views > 0:
        K, d, Q = 128, 896, 4
        di = inputs.decode_inputs(P=8, in_dim=F, seed=1)
        bf = lambda bits: torch.from_numpy(bits.view(np.int16)).to(dev).view(torch.bfloat16)
        dec = legs.make_decoder([bf(w) for w in di.weights], [torch.from_numpy(b).to(dev) for b in di.biases])
        codebook, queries = bf(di.codebook), bf(di.queries)
        probs = torch.empty((P, K), dtype=torch.bfloat16, device=dev)
        decoded = torch.empty((P, d), dtype=torch.bfloat16, device=dev)
        rel = torch.empty((P, Q), dtype=torch.float32, device=dev)
        dec_ws = torch.empty(legs.legs_decode_workspace_bytes(dec, d), dtype=torch.uint8, device=dev)
        rel_ws = torch.empty(legs.legs_relevancy_workspace_bytes(K, Q), dtype=torch.uint8, device=dev)
        legs.legs_decode_prepare(ctx, dec, codebook, dec_ws)
        legs.legs_relevancy_prepare(ctx, codebook, di.d_clip, queries, rel_ws)
        ccams = [legs.make_camera(c) for c in cams]
        t4 = []
        for k in range(2 + 5):
            flush.fill_(k)
            a0, a1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a0.record()
            for v, cc in enumerate(ccams):
                r.cam = cc
                one(None, legs.LEGS_BWD_ACCUMULATE if v else 0)
                legs.legs_decode_semantics_packed(ctx, r.sem_bf16, dec, d, probs, decoded, dec_ws)
                legs.legs_relevancy_packed(ctx, probs, K, Q, rel, rel_ws)
            a1.record()
            torch.cuda.synchronize()
            if k >= 2:
                t4.append(a0.elapsed_time(a1))
        t4 = float(np.mean(t4))
        out["step"] = dict(views=len(ccams), ms=round(t4, 4), mpix_s=round(P * len(ccams) / t4 / 1e3, 1), D_per_view=[int(x) for x in Ds],
                           what="per view: S1-S7 (gradients accumulated over the views) + decode (in_dim = F -> 64 -> 128, d = 896) + relevancy")
    return out


def run_gpu(args):
    import torch
    import torch.distributed as dist
    from paper_2311_18482_b200 import binding as legs

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    nccl_log = None
    if world > 1:
        if rank == 0 and "NCCL_DEBUG" not in os.environ:
            # the communicator line (rank count, transport) goes to a file, not to stdout (stdout carries the one JSON line)
            nccl_log = f"/tmp/legs_nccl_init_{os.getpid()}.log"
            os.environ.update(NCCL_DEBUG="INFO", NCCL_DEBUG_SUBSYS="INIT", NCCL_DEBUG_FILE=nccl_log)
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    ctx = legs.Context(local_rank)

    scene, wname = workload(args.small)
    cam = view_for_rank(scene, rank)
    W, H, F = cam.width, cam.height, scene.sem_dim
    P = W * H
    CH = inputs.channels(F)
    g = legs.Gaussians.from_scene(scene, dev)
    upstream_h = torch.from_numpy(inputs.upstream_gradient(scene, 0)).pin_memory()
    upstream = upstream_h.to(dev)
    di = inputs.decode_inputs(P=8, seed=1)   # configs[3] decoder weights, codebook and queries
    bf = lambda bits: torch.from_numpy(bits.view(np.int16)).to(dev).view(torch.bfloat16)
    dec = legs.make_decoder([bf(w) for w in di.weights], [torch.from_numpy(b).to(dev) for b in di.biases])
    codebook, queries = bf(di.codebook), bf(di.queries)
    K, d, Q = 128, 896, 4

    # capacity: one sync outside the timed region (the call a user makes once per scene/camera family)
    probe = legs.Renderer(ctx, g, cam, capacity=16)
    legs.legs_preprocess(ctx, g, probe.cam, probe.frame)
    D = legs.legs_read_num_instances(ctx, probe.frame)
    del probe
    r = legs.Renderer(ctx, g, cam, capacity=int(D * 1.02) + 1024, want_keys=False, want_bf16=True)
    if os.environ.get("LEGS_BENCH_NO_MASKS"):      # measurement switch: backward recomputes the warp-block masks
        r.block_masks = None
    grads = legs.Grads(g, dev)
    probs = torch.empty((P, K), dtype=torch.bfloat16, device=dev)
    decoded = torch.empty((P, d), dtype=torch.bfloat16, device=dev)
    rel = torch.empty((P, Q), dtype=torch.float32, device=dev)
    dec_ws = torch.empty(legs.legs_decode_workspace_bytes(dec, d), dtype=torch.uint8, device=dev)
    rel_ws = torch.empty(legs.legs_relevancy_workspace_bytes(K, Q), dtype=torch.uint8, device=dev)
    r.bwd_ws = torch.empty(legs.legs_backward_workspace_bytes(g.n, F), dtype=torch.uint8, device=dev)
    order = torch.empty(r.ntiles, dtype=torch.int32, device=dev)   # heavy tiles first (legs_tile_order, timed inside render_forward)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)   # > 126 MB L2
    # decoder weights, codebook and queries are fixed across frames: their packing (B units, Gram matrix) is done once
    legs.legs_decode_prepare(ctx, dec, codebook, dec_ws)
    legs.legs_relevancy_prepare(ctx, codebook, di.d_clip, queries, rel_ws)

    stage_names = ["preprocess", "bin_and_sort", "render_forward", "render_backward", "decode_semantics", "relevancy"]
    if world > 1:
        stage_names.append("grad_allreduce")
    NS = len(stage_names)

    def step(events=None):
        def mark(i):
            if events is not None:
                events[i].record()
        mark(0)
        legs.legs_preprocess(ctx, g, r.cam, r.frame); mark(1)
        legs.legs_bin_and_sort(ctx, r.frame, r.cam, g.n, r.capacity, None, r.vals_sorted, r.ranges, r.sort_ws); mark(2)
        legs.legs_tile_order(ctx, r.ranges, order); legs.legs_render_forward(ctx, g, r.cam, r.frame, r.vals_sorted, r.ranges, r.out, r.n_contrib, r.sem_bf16, r.block_masks, order); mark(3)
        legs.legs_render_backward(ctx, g, r.cam, r.frame, r.vals_sorted, r.ranges, r.out, r.n_contrib, upstream, 0, grads,
                                  r.bwd_ws, r.block_masks, order); mark(4)
        # by-view split: the one exchange step, a sum of the parameter gradients over the views. Issued right after S7 on
        # NCCL's own stream (async_op) so that it runs under decode + relevancy, which do not read the gradients; the step's
        # last stage is the wait = the all-reduce time that stays exposed.
        work = dist.all_reduce(grads.flat, op=dist.ReduceOp.SUM, async_op=True) if world > 1 else None
        legs.legs_decode_semantics_packed(ctx, r.sem_bf16, dec, d, probs, decoded, dec_ws); mark(5)
        legs.legs_relevancy_packed(ctx, probs, K, Q, rel, rel_ws); mark(6)
        if work is not None:
            work.wait(); mark(7)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(args.warmup, 3)):
        flush.fill_(1)
        step()
    barrier()
    # work counters for the ALU rooflines (measurement variant of the forward kernel, outside the timed region)
    counters = torch.zeros(4, dtype=torch.int64, device=dev)
    legs.legs_render_forward_stats(ctx, g, r.cam, r.frame, r.vals_sorted, r.ranges, r.out, r.n_contrib, counters)
    torch.cuda.synchronize()
    P_ek, P_b, I_f, P_e = [int(x) for x in counters.cpu().numpy()]   # examined by the kernel, blended, staged, plain walk
    n_vis = int((r.frame.tiles_touched > 0).sum().item())
    rect = r.frame.rect.view(-1, 4)
    n_rows = int(((rect[:, 3] - rect[:, 1]) * (r.frame.tiles_touched > 0)).sum().item())   # (Gaussian, tile row) entries

    # ---- timed region: K steps, device events per step (L2 flushed between steps, outside the event pairs)
    ev = [[torch.cuda.Event(enable_timing=True) for _ in range(NS + 1)] for _ in range(args.steps)]
    sampler = ClockSampler(local_rank) if rank == 0 else None
    if sampler:
        sampler.wait_first()
    launches0 = ctx.launches
    barrier()
    t_begin = time.monotonic()
    for k in range(args.steps):
        flush.fill_(k & 0xff)
        step(ev[k])
    barrier()
    t_end = time.monotonic()
    launches = ctx.launches - launches0
    step_ms = [e[0].elapsed_time(e[NS]) for e in ev]
    stage_ms = np.array([[e[i].elapsed_time(e[i + 1]) for i in range(NS)] for e in ev]).mean(0)
    t_local = float(np.sum(step_ms)) / 1e3
    if world > 1:
        tt = torch.tensor([t_local], dtype=torch.float64, device=dev)
        dist.all_reduce(tt, op=dist.ReduceOp.MAX)
        t_max = float(tt.item())
    else:
        t_max = t_local
    agg = aggregate(P * args.steps, t_local, world, (lambda t: t_max))

    # ---- the peaks the ALU rooflines divide by, measured in this run with the clock sampler still on
    alu = measure_alu_peaks(legs, ctx, torch)
    t_peaks_end = time.monotonic()
    clocks = sampler.stop(t_begin, t_end) if sampler else None
    clocks_peaks = None
    if sampler:
        pk_samples = [float(x.split(",")[0]) for (t, x) in sampler.samples if t_end < t <= t_peaks_end + 0.03 and x.split(",")[0].strip().replace(".", "").isdigit()]
        clocks_peaks = float(np.median(pk_samples)) if pk_samples else None

    # ---- S6 alone (the compositor without the projection backward): same launches, measurement flag
    s6_ms = []
    for k in range(3 + 10):
        flush.fill_(k)
        a0, a1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a0.record()
        legs.legs_render_backward(ctx, g, r.cam, r.frame, r.vals_sorted, r.ranges, r.out, r.n_contrib, upstream,
                                  legs.LEGS_BWD_COMPOSITE_ONLY, grads, r.bwd_ws, r.block_masks, order)
        a1.record()
        torch.cuda.synchronize()
        if k >= 3:
            s6_ms.append(a0.elapsed_time(a1))
    s6_ms = float(np.mean(s6_ms))

    # ---- outside the step: configs[3] at its own size (1920x1080 rows of N(0,1) features), decode + relevancy
    dec3 = None
    if not args.small:
        P3 = 1920 * 1080
        feat3 = torch.randn((P3, 8), device=dev).to(torch.bfloat16)
        probs3 = torch.empty((P3, K), dtype=torch.bfloat16, device=dev)
        decoded3 = torch.empty((P3, d), dtype=torch.bfloat16, device=dev)
        rel3 = torch.empty((P3, Q), dtype=torch.float32, device=dev)
        t3 = []
        for k in range(3 + 10):
            flush.fill_(k)
            a0, a1, a2 = (torch.cuda.Event(enable_timing=True) for _ in range(3))
            a0.record()
            legs.legs_decode_semantics_packed(ctx, feat3, dec, d, probs3, decoded3, dec_ws)
            a1.record()
            legs.legs_relevancy_packed(ctx, probs3, K, Q, rel3, rel_ws)
            a2.record()
            torch.cuda.synchronize()
            if k >= 3:
                t3.append((a0.elapsed_time(a1), a1.elapsed_time(a2)))
        t3 = np.array(t3).mean(0)
        fl3 = 2.0 * P3 * (8 * 64 + 64 * K + K * d)
        by3 = P3 * (2 * 8 + 2 * K + 2 * d)
        dec3 = dict(P=P3, decode_ms=round(float(t3[0]), 4), relevancy_ms=round(float(t3[1]), 4),
                    decode_tflops=round(fl3 / (t3[0] * 1e-3) / 1e12, 1), decode_gb_s=round(by3 / (t3[0] * 1e-3) / 1e9, 1))
        # the paper's own decoder shape (Table 3: 8 -> 128 -> 256 -> N): the one shape where the tensor pipe,
        # not the HBM write, should bind (181 248 MAC / pixel); and S11 from the decoded map (input_is_probs = 0)
        di_t3 = inputs.decode_inputs(P=8, seed=1, hidden=(128, 256), bias_sigma=0.1)
        dec_t3 = legs.make_decoder([bf(w) for w in di_t3.weights], [torch.from_numpy(b).to(dev) for b in di_t3.biases])
        ws_t3 = torch.empty(legs.legs_decode_workspace_bytes(dec_t3, d), dtype=torch.uint8, device=dev)
        legs.legs_decode_prepare(ctx, dec_t3, codebook, ws_t3)
        tt3 = []
        for k in range(3 + 10):
            flush.fill_(k)
            a0, a1, a2 = (torch.cuda.Event(enable_timing=True) for _ in range(3))
            a0.record()
            legs.legs_decode_semantics_packed(ctx, feat3, dec_t3, d, probs3, decoded3, ws_t3)
            a1.record()
            legs.legs_relevancy_decoded(ctx, decoded3, di.d_clip, queries, rel3)
            a2.record()
            torch.cuda.synchronize()
            if k >= 3:
                tt3.append((a0.elapsed_time(a1), a1.elapsed_time(a2)))
        tt3 = np.array(tt3).mean(0)
        fl_t3 = 2.0 * P3 * (8 * 128 + 128 * 256 + 256 * K + K * d)
        pk_ = peaks()
        dec3["table3"] = dict(shape="8->128->256->128 (PAPER.md Table 3), d = 896", decode_ms=round(float(tt3[0]), 4),
                              decode_tflops=round(fl_t3 / (tt3[0] * 1e-3) / 1e12, 1),
                              frac_bf16_peak=round(fl_t3 / (tt3[0] * 1e-3) / 1e12 / pk_["bf16"], 4),
                              decode_gb_s=round(by3 / (tt3[0] * 1e-3) / 1e9, 1),
                              frac_hbm=round(by3 / (tt3[0] * 1e-3) / 1e9 / pk_["hbm_gbs"], 4),
                              tensor_roofline_ms=round(fl_t3 / (pk_["bf16"] * 1e12) * 1e3, 4),
                              hbm_roofline_ms=round(by3 / (pk_["hbm_gbs"] * 1e9) * 1e3, 4))
        by_rd = P3 * (2 * di.d_clip + 4 * Q)
        dec3["relevancy_from_decoded"] = dict(ms=round(float(tt3[1]), 4), gb_s=round(by_rd / (tt3[1] * 1e-3) / 1e9, 1),
                                              frac_hbm=round(by_rd / (tt3[1] * 1e-3) / 1e9 / pk_["hbm_gbs"], 4),
                                              note="legs_relevancy_decoded: reads the first d_clip columns of the decoded map (1 KB / pixel)")
        del feat3, probs3, decoded3, rel3, ws_t3

    # ---- outside the step: the widening rows, timed on the rendered maps / the gradients of the step
    index_map = torch.randint(0, K, (P,), dtype=torch.int32, device=dev)
    dL_loss = torch.zeros_like(r.out)
    dw = [torch.zeros(tuple(w.shape), dtype=torch.float32, device=dev) for w in di.weights]
    dbs = [torch.zeros(tuple(b.shape), dtype=torch.float32, device=dev) for b in di.biases]
    loss_buf = torch.zeros(3, dtype=torch.float32, device=dev)
    loss_ws = torch.empty(legs.legs_loss_workspace_bytes(dec, P), dtype=torch.uint8, device=dev)
    params = [g.t[k] for k in ("means", "scales", "quats", "opacities", "sh", "sem", "unc")]
    pgrads = [grads.dmeans, grads.dscales, grads.dquats, grads.dopacities, grads.dsh, grads.dsem, grads.dunc]
    adam_m = [torch.zeros_like(t) for t in params]
    adam_v = [torch.zeros_like(t) for t in params]
    saved = [t.clone() for t in params]
    den = (torch.zeros(g.n, device=dev), torch.zeros(g.n, dtype=torch.int32, device=dev), torch.zeros(g.n, dtype=torch.int32, device=dev))
    loss_ms, adam_ms, dens_ms = [], [], []
    for k in range(3 + 10):
        flush.fill_(k)
        a = [torch.cuda.Event(enable_timing=True) for _ in range(4)]
        a[0].record()
        legs.legs_semantic_loss(ctx, r.out, index_map, dec, 1.0, 0.1, dL_loss, dw, dbs, loss_buf, loss_ws)
        a[1].record()
        legs.legs_adam_step(ctx, params, pgrads, adam_m, adam_v, k + 1)
        a[2].record()
        legs.legs_density_stats(ctx, grads.dmean2d, r.frame.radius, *den)
        a[3].record()
        torch.cuda.synchronize()
        if k >= 3:
            loss_ms.append(a[0].elapsed_time(a[1])); adam_ms.append(a[1].elapsed_time(a[2])); dens_ms.append(a[2].elapsed_time(a[3]))
    for t, sv in zip(params, saved):
        t.copy_(sv)       # the e2e pass below renders the original scene again
    # quantisation search (8(f) item 2) on one frame of synthetic 896-dim features: [P, 896] x [896, 128]
    quant = None
    if not args.small:
        qi = inputs.quantize_inputs(P=4096, n_codes=K, d=d, d_clip=di.d_clip, seed=5)
        reps = (P + 4095) // 4096
        qfeat = bf(qi.features).repeat(reps, 1)[:P].contiguous()      # the 4096 synthetic rows tiled over the frame
        qcode = bf(qi.codebook)
        qidx = torch.empty(P, dtype=torch.int32, device=dev)
        qr, qp_, ql = torch.zeros(K, device=dev), torch.zeros(K, device=dev), torch.zeros(4, device=dev)
        qms = []
        for k in range(3 + 10):
            flush.fill_(k)
            a0, a1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a0.record()
            legs.legs_quantize(ctx, qfeat, qcode, di.d_clip, 0.5, 1.0, 0.5, qidx, qr, qp_, ql)
            a1.record()
            torch.cuda.synchronize()
            if k >= 3:
                qms.append(a0.elapsed_time(a1))
        qms = float(np.mean(qms))
        qbytes = P * (2 * d + 4)
        quant = dict(ms=round(qms, 4), gb_s=round(qbytes / (qms * 1e-3) / 1e9, 1), frac_hbm=round(qbytes / (qms * 1e-3) / 1e9 / peaks()["hbm_gbs"], 4),
                     tflops=round(2.0 * P * d * K / (qms * 1e-3) / 1e12, 1))
        del qfeat, qidx
    loss_ms, adam_ms, dens_ms = float(np.mean(loss_ms)), float(np.mean(adam_ms)), float(np.mean(dens_ms))
    # the loss head on the paper's Table 3 decoder (8 -> 128 -> 256 -> N), forward + reverse mode
    loss_t3 = None
    if not args.small:
        di_l3 = inputs.decode_inputs(P=8, seed=1, hidden=(128, 256), bias_sigma=0.1)
        dec_l3 = legs.make_decoder([bf(w) for w in di_l3.weights], [torch.from_numpy(b).to(dev) for b in di_l3.biases])
        dw3 = [torch.zeros(tuple(w.shape), dtype=torch.float32, device=dev) for w in di_l3.weights]
        db3 = [torch.zeros(tuple(b.shape), dtype=torch.float32, device=dev) for b in di_l3.biases]
        ws_l3 = torch.empty(legs.legs_loss_workspace_bytes(dec_l3, P), dtype=torch.uint8, device=dev)
        l3 = []
        for k in range(3 + 10):
            flush.fill_(k)
            a0, a1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a0.record()
            legs.legs_semantic_loss(ctx, r.out, index_map, dec_l3, 1.0, 0.1, dL_loss, dw3, db3, loss_buf, ws_l3)
            a1.record()
            torch.cuda.synchronize()
            if k >= 3:
                l3.append(a0.elapsed_time(a1))
        l3 = float(np.mean(l3))
        fl_l3 = 2.0 * P * (8 * 128 + 3 * 128 * 256 + 3 * 256 * K)      # forward, dX and dW of the two tensor-core layers + layer 0
        loss_t3 = dict(ms=round(l3, 4), tflops=round(fl_l3 / (l3 * 1e-3) / 1e12, 1),
                       frac_bf16_peak=round(fl_l3 / (l3 * 1e-3) / 1e12 / peaks()["bf16"], 4))
        del ws_l3
    # adaptive spatial smoothing (8(f) item 3): the Table 4 MLP over all n Gaussians, forward + reverse mode
    swb, sbias = inputs.smooth_mlp_inputs(sem_dim=F, seed=3)
    sw = [bf(w) for w in swb]
    sb = [torch.from_numpy(b).to(dev) for b in sbias]
    sdw = [torch.zeros(tuple(w.shape), dtype=torch.float32, device=dev) for w in swb]
    sdb = [torch.zeros(tuple(b.shape), dtype=torch.float32, device=dev) for b in sbias]
    sds = torch.zeros((g.n, F), dtype=torch.float32, device=dev)
    sloss = torch.zeros(4, dtype=torch.float32, device=dev)
    pos = (g.t["means"] / 50.0).contiguous()
    smooth_ms = []
    for k in range(3 + 10):
        flush.fill_(k)
        a0, a1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a0.record()
        legs.legs_smooth_loss(ctx, pos, g.t["sem"], g.t["unc"], sw, sb, 0.1, 1.0, False, sds, sdw, sdb, sloss)
        a1.record()
        torch.cuda.synchronize()
        if k >= 3:
            smooth_ms.append(a0.elapsed_time(a1))
    smooth_ms = float(np.mean(smooth_ms))
    smooth_flops = 2.0 * g.n * (128 * 128 * 2 * 3 + 128 * F * 3 + 3 * 128 * 2)     # fwd + dX + dW of the two 128x128 layers, ends
    del sds, pos
    n_param = sum(t.numel() for t in params)
    del dL_loss, adam_m, adam_v, saved

    # ---- e2e: same calls, host (pinned) inputs copied in and results copied out inside the timed region, every step.
    # Frames are streamed the way a user of the library would: two device slots, copies on their own streams, so the
    # H2D copy of step k+1 and the D2H copy of step k-1 overlap the kernels of step k (PCIe is full duplex).
    host_in = {k: v.cpu().pin_memory() for k, v in g.t.items()}
    out_keys = ("dmeans", "dscales", "dquats", "dopacities", "dsh", "dsem", "dunc", "dmean2d")

    class Slot:
        def __init__(self, first):
            if first:
                self.g, self.r, self.grads, self.upstream = g, r, grads, upstream
                self.probs, self.decoded, self.rel = probs, decoded, rel
            else:
                self.g = legs.Gaussians(*[g.t[k].clone() for k in ("means", "scales", "quats", "opacities", "sh", "sem", "unc")],
                                        g.sh_degree)
                self.r = legs.Renderer(ctx, self.g, cam, capacity=r.capacity, want_keys=False, want_bf16=True)
                self.r.bwd_ws = torch.empty_like(r.bwd_ws)
                self.grads = legs.Grads(self.g, dev)
                self.upstream = torch.empty_like(upstream)
                self.probs, self.decoded, self.rel = torch.empty_like(probs), torch.empty_like(decoded), torch.empty_like(rel)
            self.host_out = dict(out=torch.empty((H, W, CH), dtype=torch.float32).pin_memory(),
                                 rel=torch.empty((P, Q), dtype=torch.float32).pin_memory(),
                                 **{k: torch.empty_like(getattr(self.grads, k), device="cpu").pin_memory() for k in out_keys})
            self.in_ready, self.computed, self.copied = (torch.cuda.Event() for _ in range(3))

        def run(self):
            s = self
            legs.legs_preprocess(ctx, s.g, s.r.cam, s.r.frame)
            legs.legs_bin_and_sort(ctx, s.r.frame, s.r.cam, s.g.n, s.r.capacity, None, s.r.vals_sorted, s.r.ranges, s.r.sort_ws)
            legs.legs_tile_order(ctx, s.r.ranges, order)
            legs.legs_render_forward(ctx, s.g, s.r.cam, s.r.frame, s.r.vals_sorted, s.r.ranges, s.r.out, s.r.n_contrib, s.r.sem_bf16,
                                     s.r.block_masks, order)
            legs.legs_render_backward(ctx, s.g, s.r.cam, s.r.frame, s.r.vals_sorted, s.r.ranges, s.r.out, s.r.n_contrib,
                                      s.upstream, 0, s.grads, s.r.bwd_ws, s.r.block_masks, order)
            legs.legs_decode_semantics_packed(ctx, s.r.sem_bf16, dec, d, s.probs, s.decoded, dec_ws)
            legs.legs_relevancy_packed(ctx, s.probs, K, Q, s.rel, rel_ws)
            if world > 1:
                dist.all_reduce(s.grads.flat, op=dist.ReduceOp.SUM)

    slots = [Slot(True), Slot(False)]
    h2d = sum(v.numel() * v.element_size() for v in host_in.values()) + upstream_h.numel() * 4
    d2h = sum(v.numel() * v.element_size() for v in slots[0].host_out.values())
    st_in, st_run, st_out = torch.cuda.Stream(), torch.cuda.Stream(), torch.cuda.Stream()

    def e2e_steps_run(nsteps):
        for k in range(nsteps):
            sl = slots[k & 1]
            with torch.cuda.stream(st_in):
                st_in.wait_event(sl.computed)        # the slot's previous step has consumed its inputs
                for name, v in host_in.items():
                    sl.g.t[name].copy_(v, non_blocking=True)
                sl.upstream.copy_(upstream_h, non_blocking=True)
                sl.in_ready.record(st_in)
            with torch.cuda.stream(st_run):
                st_run.wait_event(sl.in_ready)
                st_run.wait_event(sl.copied)         # the slot's previous results have left the device
                sl.run()
                sl.computed.record(st_run)
            with torch.cuda.stream(st_out):
                st_out.wait_event(sl.computed)
                sl.host_out["out"].copy_(sl.r.out, non_blocking=True)
                sl.host_out["rel"].copy_(sl.rel, non_blocking=True)
                for name in out_keys:
                    sl.host_out[name].copy_(getattr(sl.grads, name), non_blocking=True)
                sl.copied.record(st_out)

    e2e_steps = max(4, min(args.steps, 10))
    barrier()
    e2e_steps_run(2)
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(st_in)
    e2e_steps_run(e2e_steps)
    e1.record(st_out)
    barrier()
    t_e2e = e0.elapsed_time(e1) / 1e3
    if world > 1:
        tt = torch.tensor([t_e2e], dtype=torch.float64, device=dev)
        dist.all_reduce(tt, op=dist.ReduceOp.MAX)
        t_e2e = float(tt.item())
    e2e_val = P * e2e_steps * world / t_e2e / 1e6

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- rooflines: algorithmic bytes / lane-instructions per call, two work models per stage:
    # "survey" = SURVEY.md 8(d) (plain per-tile walk: P_e examined pairs; 6-pass LSD sort over the D instances) and
    # "built" = the algorithm as built (block-culled pairs P_ek; no pass over D in the binning).
    pk = peaks()
    alu_peak = alu["ffma_t_lane_instr_s"]
    n = g.n
    ntiles = math.ceil(W / 16) * math.ceil(H / 16)
    RSb = 4 * legs.record_stride(F)
    pre_bytes = n * (12 + 65) + n_vis * (12 + 16 + 4 + 192 + 4 * F + 4 + RSb)
    s7_bytes = n_vis * (240 + 4 * (10 + F)) + n_vis * (4 * (3 + 3 + 4 + 1 + 48 + F + 1 + 2))
    alg_built = {
        "preprocess": ("hbm", pre_bytes),
        # depth sort of n (histogram read + 4 passes), rect/tiles reads (counting + ranked emission), row entries (8 B
        # written once, straight into (row, depth) order; read by the chunk counts and by the expansion), one 4-byte write
        # per tile instance, ranges
        "bin_and_sort": ("hbm", n * (4 + 4 * 16 + 2 * 20) + n_rows * (8 + 8 + 8) + D * 4 + ntiles * 8),
        "render_forward": ("alu", 12 * P_ek + (4 + 3 + F + 2) * P_b),
        "render_backward_s6": ("alu", 12 * P_ek + (75 + 20) * P_b),
        "decode_semantics": ("hbm", P * (2 * 8 + 2 * K + 2 * d)),
        "relevancy": ("hbm", P * (2 * K + 4 * Q)),
    }
    alg_survey = {
        "preprocess": ("hbm", pre_bytes),
        "bin_and_sort": ("hbm", n * 12 + D * (12 + 152 + 8)),                       # S2 + S3 + S4a (6-pass LSD) + S4b
        "render_forward": ("alu", 12 * P_e + (4 + 3 + F + 2) * P_b),
        "render_backward_s6": ("alu", 12 * P_e + (75 + 20) * P_b),                  # 12 P_e + 95 P_b
        "decode_semantics": alg_built["decode_semantics"],
        "relevancy": alg_built["relevancy"],
    }
    s7_ms = float(stage_ms[3]) - s6_ms
    ms_of = {"preprocess": float(stage_ms[0]), "bin_and_sort": float(stage_ms[1]), "render_forward": float(stage_ms[2]),
             "render_backward_s6": s6_ms, "decode_semantics": float(stage_ms[4]), "relevancy": float(stage_ms[5])}

    def roof(name, model):
        bound, work = model[name]
        sec = ms_of[name] / 1e3
        if bound == "hbm":
            ach, peak, unit = work / sec / 1e9, pk["hbm_gbs"], "GB/s"
        else:
            ach, peak, unit = work / sec / 1e12, alu_peak, "T lane-instr/s"
        return dict(bound=bound, achieved=round(ach, 3), peak=round(peak, 3), unit=unit, frac=round(ach / peak, 4),
                    ms=round(ms_of[name], 4), work=int(work), roofline_ms=round(work / (peak * (1e9 if bound == "hbm" else 1e12)) * 1e3, 4))

    rooflines = {name: dict(survey=roof(name, alg_survey), built=roof(name, alg_built)) for name in ms_of}
    rooflines["project_backward_s7"] = dict(built=dict(bound="hbm", ms=round(s7_ms, 4), work=int(s7_bytes),
                                                       achieved=round(s7_bytes / (s7_ms / 1e3) / 1e9, 1), peak=pk["hbm_gbs"], unit="GB/s",
                                                       frac=round(s7_bytes / (s7_ms / 1e3) / 1e9 / pk["hbm_gbs"], 4)))
    dom = max(ms_of, key=lambda k: ms_of[k])
    kern = {"render_backward_s6": r"backward_kernel", "render_forward": r"forward_kernel", "decode_semantics": r"decode_kernel",
            "bin_and_sort": r"expand_kernel", "preprocess": r"preprocess_kernel", "relevancy": r"relevancy_kernel"}[dom]
    # Headline = the work the kernel really does: pairs it examines after its block culling (P_ek, counted on the
    # device by legs_render_forward_stats) x 12 lane-instructions + blended pairs x 95. The survey's plain-walk count (P_e) stays
    # as a secondary key; so does what the committed ncu capture says the kernel issues (32 lane slots per warp instruction).
    rf = dict(rooflines[dom]["built"])
    ncu = None if args.small else ncu_committed(kern)
    work_models = {"render_backward_s6": "as built: 12 P_ek + 95 P_b lane-instructions, P_ek = pairs examined after block culling",
                   "render_forward": "as built: 12 P_ek + (9 + F) P_b lane-instructions"}
    roofline = dict(bound=rf["bound"], achieved=rf["achieved"], peak=rf["peak"], unit=rf["unit"], frac=rf["frac"],
                    traffic=None if ncu is None else ncu["traffic"], traffic_source=None if ncu is None else ncu["source"],
                    kernel=dom, kernel_ms=rf["ms"], work=rf["work"],
                    work_model=work_models.get(dom, "as built: algorithmic bytes of the call (DESIGN.md section 6)"),
                    frac_survey_model=rooflines[dom]["survey"]["frac"],
                    survey_model="SURVEY.md 8(d): plain per-tile walk, P_e examined pairs" if rf["bound"] == "alu" else "SURVEY.md 8(d)",
                    peak_source=(pk["source"] + " (MEASURED_PEAKS.json)") if rf["bound"] == "hbm" else
                    "measured in run: FFMA-chain micro-benchmark (legs_peak_kernel)",
                    mufu_ex2_peak_t_s=alu["ex2_t_s"], mufu_floor_ms=round(P_ek / (alu["ex2_t_s"] * 1e12) * 1e3, 4))
    if ncu is not None and rf["bound"] == "alu" and ncu["warp_instructions"]:
        roofline["ncu_committed"] = dict(issue_active_pct=ncu["issue_active_pct"], warp_instructions=ncu["warp_instructions"],
                                         issued_lane_slots_over_work=round(32.0 * ncu["warp_instructions"] / rf["work"], 3))

    def path(names, label):
        ms = sum(float(stage_ms[stage_names.index(nm)]) for nm in names)
        out = dict(ms=round(ms, 4), mpix_s=round(P / ms / 1e3, 2))
        for model_name, model in (("survey", alg_survey), ("built", alg_built)):
            t = 0.0
            for nm in names:
                keys = ["render_backward_s6"] if nm == "render_backward" else [nm]
                for kk in keys:
                    bound, work = model[kk]
                    t += work / (pk["hbm_gbs"] * 1e9 if bound == "hbm" else alu_peak * 1e12)
                if nm == "render_backward":
                    t += s7_bytes / (pk["hbm_gbs"] * 1e9)
            out[f"roofline_ms_{model_name}"] = round(t * 1e3, 4)
            out[f"frac_{model_name}"] = round(t * 1e3 / ms, 4)
        return out

    fwd = path(["preprocess", "bin_and_sort", "render_forward"], "fwd")
    fwd_bwd = path(["preprocess", "bin_and_sort", "render_forward", "render_backward"], "fwd_bwd")
    dec_flops = 2.0 * P * (8 * 64 + 64 * K + K * d)
    tensor = dict(tflops=round(dec_flops / (stage_ms[4] / 1e3) / 1e12, 2), peak=pk["bf16"],
                  frac=round(dec_flops / (stage_ms[4] / 1e3) / 1e12 / pk["bf16"], 4), configs3=dec3)

    # ---- the other raster configs, one view each (configs[4] also as its whole 4-view step)
    per_config = None
    if not args.small and not args.no_per_config:
        torch.cuda.empty_cache()
        per_config = {
            "configs1": time_config(legs, ctx, torch, inputs.object_scene(), "configs[1] object scene: 100k Gaussians, 800x800, SH3, F=8+u, view 0",
                                    flush, alu_peak, pk["hbm_gbs"]),
            "configs4": time_config(legs, ctx, torch, inputs.large_scene(), "configs[4] large scene: 3M Gaussians, 1920x1080, SH3, F=16+u, view 0; step = 4 views",
                                    flush, alu_peak, pk["hbm_gbs"], step_views=4),
        }

    cpu = None
    if not args.no_cpu_baseline:
        cpu = oracle_sample_throughput(scene, scene.cameras[0], args.ref_sample)
        cpu["configs0"] = oracle_small_configs()
        if not args.no_oracle_configs1:
            cpu["configs1_whole_frame"] = oracle_configs1_whole_frame()
    line = dict(metric=METRIC, value=round(agg["mpix_s"], 2), unit=UNIT, n_gpus=world, steps=args.steps, warmup=max(args.warmup, 3),
                ms_per_step=round(float(np.mean(step_ms)), 4), higher_is_better=True, scaling="weak", vs_baseline=None,
                dtype="f32", data="synthetic",
                config=dict(workload=wname, step="S1-S7 + S9-S11: preprocess, bin_and_sort, render_forward, render_backward, "
                            "decode_semantics, relevancy" + (", gradient all-reduce" if world > 1 else ""),
                            step_notes="render_forward includes legs_tile_order (one 19 us launch: compositor CTAs start with the longest tile "
                                       "lists; both compositors use it); decode and relevancy run on weights / codebook / Gram matrix packed once before the timed "
                                       "region (legs_*_packed: the inference path; a training step would repack per iteration); the "
                                       "upstream gradient of render_backward is a fixed random map: the semantic loss head that "
                                       "produces it is timed apart under next_rows, not inside the step",
                            parallelism=f"by view: {world} replicas, one view each, one NCCL all-reduce of the gradients per step, overlapped with decode + relevancy (stages_ms.grad_allreduce = exposed time)" if world > 1 else "single GPU",
                            nccl_init=nccl_init_lines(nccl_log),
                            l2="flushed between steps (256 MB write)", D=D, n_visible=n_vis, row_entries=n_rows,
                            examined_pairs_plain_walk=P_e, examined_pairs_after_block_culling=P_ek, blended_pairs=P_b,
                            staged_list_entries=I_f, num_sms=ctx.num_sms),
                fwd=fwd, fwd_bwd=fwd_bwd, per_config=per_config,
                stages_ms={k: round(float(v), 4) for k, v in zip(stage_names, stage_ms)},
                backward_split_ms=dict(s6_compositor=round(s6_ms, 4), s7_projection=round(s7_ms, 4)),
                roofline=roofline, rooflines=rooflines, measured_alu_peaks=dict(alu, sm_mhz_during=clocks_peaks), decode_tensor=tensor,
                next_rows=dict(semantic_loss_ms=round(loss_ms, 4), semantic_loss_table3=loss_t3, adam_step_ms=round(adam_ms, 4),
                               adam_gb_s=round(n_param * 28 / (adam_ms * 1e-3) / 1e9, 1), density_stats_ms=round(dens_ms, 4), quantize=quant,
                               smooth_loss=dict(ms=round(smooth_ms, 4), tflops=round(smooth_flops / (smooth_ms * 1e-3) / 1e12, 1),
                                                frac_bf16_peak=round(smooth_flops / (smooth_ms * 1e-3) / 1e12 / peaks()["bf16"], 4)),
                               note="widening rows (SURVEY.md 8(f)) timed on the step's outputs; not part of the step"),
                e2e=dict(value=round(e2e_val, 2), unit=UNIT, h2d_bytes_per_step=int(h2d), d2h_bytes_per_step=int(d2h),
                         ms_per_step=round(t_e2e / e2e_steps * 1e3, 3),
                         note="two device slots; H2D, kernels and D2H on three streams; copied out: image record, relevancy map, all "
                              "gradients. The decoded feature map (3.05 GB) and the probabilities stay on the device"),
                gpu_launches=int(launches), clocks=clocks,
                cpu_baseline=None if cpu is None else {k: cpu[k] for k in ("value", "unit", "cores", "kind", "sample", "configs0",
                                                                            "configs1_whole_frame") if k in cpu})
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="legs", choices=["legs", "reference"])
    ap.add_argument("--small", action="store_true", help="reduced workload (debugging only; not the benchmark)")
    ap.add_argument("--ref-sample", type=int, default=2048, help="pixels per oracle sample")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-oracle-configs1", action="store_true",
                    help="skip the oracle's one whole configs[1] frame (about 20 s on the 16 host cores of the B200 box)")
    ap.add_argument("--no-per-config", action="store_true", help="skip the configs[1] / configs[4] timings (per_config)")
    ap.add_argument("--dry-host", action="store_true",
                    help="N > 1 plumbing only, on CPU with gloo (spawn, views, gradient all-reduce, one JSON line); no kernels")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    elif args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        sys.exit(relaunch_under_torchrun(args, sys.argv[1:]))
    elif args.dry_host:
        run_dry_host(args)
    else:
        run_gpu(args)


if __name__ == "__main__":
    main()
