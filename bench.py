#!/usr/bin/env python
"""bench.py -- throughput of the neural-OIT hot path on B200 (contract: see DESIGN.md section 7).

`metric` / `value` are BASELINE.json's: Mpixels/s (and fragments/s, % of the HBM roofline) of the
neural-OIT resolve at 1080p -- the plain fused resolve (S1-S5, `noit_resolve`) of the 1080p
high-depth-complexity workload (BASELINE.json configs[2], "cfg3"): value = P / its mean CUDA-event
time, `ms_per_step` = that time.  It is timed inside the step loop below, so every launch finds
the L2 holding other kernels' data (and its 647 MB of inputs exceed the 126 MB L2 anyway).

One STEP = one pass of the whole hot path over that frame:
   1. noit_resolve   plain fused resolve of the frame (S1-S5)          <- dominant kernel, `value`
   2. noit_quadtree  colour-variance tiles of its result (S6)
      + noit_quadtree_balance  2:1 tile consistency, histogram, demand index, Eq. 2 (NEXT-1)
   3. noit_resolve   adaptive resolve guided by those tiles (S7)
   4. noit_reproject previous result under a small camera motion (S8)
   5. noit_resolve   fallback resolve of the rejected pixels (S9)
The whole step (three output frames) is reported beside it as `step_*` (eager, serial CUDA graph,
forked CUDA graph), every kernel of the step has a line in `roofline_all`.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--scaling weak|strong]
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

BG = (0.2, 0.3, 0.4)
WORKLOAD = "cfg3: 1920x1080, 512 ellipses, mean 24 / max 128 fragments per pixel, RGBA fp16, bf16 weights"
METRIC = "Mpixels/s and fragments/s of neural OIT resolve at 1080p; % of HBM roofline"
# `config` is the same dict in both arms when both run the whole frame (the driver compares them)
WHAT_IS_TIMED = "the plain fused resolve (S1-S5) of the whole frame, one call per step"
L2_NOTE = "inputs (647 MB) larger than L2 (126 MB); no flush"


def peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        try:
            d = json.load(open(path))
            return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """nvidia-smi clocks + throttle reasons sampled DURING the timed region."""
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.samples, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "20"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            threading.Thread(target=self._read, daemon=True).start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.samples.append(line.strip())

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for s in self.samples:
            f = [x.strip() for x in s.split(",")]
            try:
                sm.append(float(f[0]))
                mx.append(float(f[1]))
            except (ValueError, IndexError):
                continue
            for n, v in zip(names, f[2:6]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


def camera_shift_matrix(W: int, H: int) -> np.ndarray:
    """Small camera motion for step 4: NDC translation of (1.5, 0.5) pixels, depth untouched."""
    M = np.eye(4, dtype=np.float64)
    M[0, 3] = 2.0 * 1.5 / W
    M[1, 3] = 2.0 * 0.5 / H
    return M.astype(np.float32)


def resolve_traffic():
    """(dram bytes per launch of the plain resolve, source file): the newest committed ncu capture
    profiles/rNN_resolve_ncu.json.txt (one `ncu --set full` launch; re-captured when the kernel
    changes -- the command is in the .md of the same name)."""
    import glob
    for path in sorted(glob.glob(os.path.join(ROOT, "profiles", "r*_resolve_ncu.json.txt")), reverse=True):
        try:
            d = json.load(open(path))
            return int(d["dram_bytes_read"]) + int(d["dram_bytes_write"]), os.path.relpath(path, ROOT)
        except Exception:
            continue
    return None, None


def step_bytes(fbh, half, quarter, lod_of_pixel, rejected, F_rejected):
    """Algorithmic bytes of every kernel of the step (SURVEY 8(d) formulas; fp16 colours)."""
    P, F = fbh.num_pixels, fbh.num_fragments
    W, H = fbh.width, fbh.height
    n = np.diff(fbh.offsets.astype(np.int64))
    coarse = lod_of_pixel > 0
    b = {"resolve": resolve_bytes(P, F, 8, 2, True)}
    b["quadtree"] = 16 * P + 4 * ((W + 63) // 64) * ((H + 63) // 64) + ((W + 7) // 8) * ((H + 7) // 8) + 16
    b["balance"] = 8 * ((W + 63) // 64) * ((H + 63) // 64) + ((W + 7) // 8) * ((H + 7) // 8) + 28
    # adaptive: lod-0 pixels read their whole list; lod>0 pixels only their depths + the winner's
    # colour; the coarse lists of coarse leaves are read once, plus their offsets; one image out
    ad = 4 * (P + 1) + 16 * P + 12 * int(n[~coarse].sum()) + 4 * int(n[coarse].sum()) + 8 * int((n[coarse] > 0).sum())
    for lod, cb in ((1, half), (2, quarter)):
        yy, xx = np.divmod(np.arange(cb.num_pixels), cb.width)
        fy, fx = np.minimum(yy << lod, H - 1), np.minimum(xx << lod, W - 1)
        used = lod_of_pixel[fy * W + fx] == lod
        cn = np.diff(cb.offsets.astype(np.int64))
        ad += 12 * int(cn[used].sum()) + 4 * int(used.sum())
    b["adaptive"] = ad
    # reproject: cur depth + gathered prev depth and prev trans; trans, depth, final, accept out
    b["reproject"] = 4 * P + 4 * P + 16 * P + (16 + 4 + 16 + 1) * (P - rejected) + P + 4 * rejected
    b["fallback"] = 4 * rejected + 8 * rejected + 12 * F_rejected + 36 * rejected
    return b


def resolve_bytes(P: int, F: int, color_bytes: int, n_images: int, depth1: bool) -> int:
    """Algorithmic bytes of the fused resolve: offsets + fragments + outputs."""
    return 4 * (P + 1) + F * (4 + color_bytes) + 16 * P * n_images + (4 * P if depth1 else 0)


def dist_setup(n_gpus: int, backend: str):
    import torch.distributed as dist
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group(backend=backend)
        return dist, dist.get_rank(), world
    return None, 0, 1


def max_over_ranks(dist, value: float, device) -> float:
    import torch
    if dist is None:
        return value
    t = torch.tensor([value], dtype=torch.float64, device="cpu" if dist.get_backend() == "gloo" else device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def run_dryrun(args):
    """CPU/gloo exercise of the N>1 plumbing (tests/test_abi.py): no GPU work, no numbers."""
    import torch
    dist, rank, world = dist_setup(args.gpus, "gloo")
    t = torch.ones(1)
    if dist is not None:
        dist.barrier()
        dist.all_reduce(t)
    ms = max_over_ranks(dist, 1.0 + rank, "cpu")
    if rank == 0:
        print(json.dumps({"metric": METRIC, "value": None, "n_gpus": world, "dryrun": True,
                          "scaling": "weak", "ranks_seen": int(t.item()), "ms_per_step": ms}))
    if dist is not None:
        dist.destroy_process_group()


def run_reference(args):
    """`--impl reference`: the oracle, as it stands, on the host cores, same metric as the product
    arm: each step = the plain resolve (S1-S5) of the cfg3 frame, or of a 256-row band of it when a
    whole frame takes more than 4 s on this host (bounded sample)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import noit_scenes
    import oracle
    sc = noit_scenes.cfg3(0)
    w_eff = oracle.effective_weights(sc.weights, sc.mlp_precision)
    fbh = sc.full
    t0 = time.perf_counter()
    oracle.resolve(fbh, w_eff, BG)
    what = WHAT_IS_TIMED
    if time.perf_counter() - t0 > 4.0:
        fbh = fbh.rows(384, 640)
        what = "the plain resolve (S1-S5) of rows 384..639 of the frame (bounded sample), one call per step"
    for _ in range(args.warmup):
        oracle.resolve(fbh, w_eff, BG)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle.resolve(fbh, w_eff, BG)
    dt = time.perf_counter() - t0
    P, F = fbh.num_pixels, fbh.num_fragments
    value = P * args.steps / dt / 1e6
    cores = oracle.num_threads()
    sample = f"plain resolve of {fbh.height} rows of the cfg3 frame ({P} pixels, {F} fragments) per step"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": "Mpixels/s", "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic",
        "config": {"workload": WORKLOAD, "pixels": P, "fragments": F, "what_is_timed": what, "l2": L2_NOTE,
                   "sharding": "none"},
        "fragments_per_s": F * args.steps / dt,
        "cpu_baseline": {"value": value, "unit": "Mpixels/s", "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": "Mpixels/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


def run_ours(args):
    import torch

    import noit_scenes
    import paper_2606_16747_b200 as noit

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device and no CPU fallback (use --impl reference for the oracle)")
    local = int(os.environ.get("LOCAL_RANK", "0"))
    # NOIT_BENCH_ONE_GPU=1: functional check of the N > 1 code path on a box with one GPU (every rank on
    # cuda:0, gloo instead of NCCL, which refuses two ranks on one device) -- its numbers mean nothing
    one_gpu = bool(os.environ.get("NOIT_BENCH_ONE_GPU"))
    if one_gpu:
        local = 0
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    dist, rank, world = dist_setup(args.gpus, "gloo" if one_gpu else "nccl")

    if args.scaling == "strong" and world > 1:
        # strong scaling: ONE cfg3 frame (seed 0) split into 64-row-aligned, fragment-balanced row
        # bands; every rank runs the whole step on its band, no data-path collective
        # (a reprojected pixel whose source row lies outside the band counts as disoccluded and is
        # resolved by S9, so no halo is exchanged)
        from paper_2606_16747_b200.sharding import shard_rows
        whole = noit_scenes.cfg3(0, coarse=True)
        bands = shard_rows(whole.full.offsets, whole.full.width, whole.full.height, world)
        y0, y1 = bands[rank]
        if y1 <= y0:
            raise SystemExit(f"bench.py: rank {rank} got an empty band ({world} ranks, {whole.full.height} rows)")
        sc = noit_scenes.Scene(f"cfg3-rows-{y0}-{y1}", whole.full.rows(y0, y1),
                               whole.half.rows(y0 // 2, (y1 + 1) // 2), whole.quarter.rows(y0 // 4, (y1 + 3) // 4),
                               whole.weights, whole.mlp_precision)
        P_job, F_job = whole.full.num_pixels, whole.full.num_fragments
        del whole
    else:
        # weak scaling: every rank resolves its own 1080p frame (seed = rank), no data-path collective
        sc = noit_scenes.cfg3(rank, coarse=True)
        P_job, F_job = sc.full.num_pixels * world, sc.full.num_fragments * world
    fbh = sc.full
    W, H, P, F = fbh.width, fbh.height, fbh.num_pixels, fbh.num_fragments
    fb, hb, qb = (noit.DeviceFragBuf.from_host(b, dev) for b in (sc.full, sc.half, sc.quarter))
    ctx = noit.Noit(sc.weights, sc.mlp_precision)
    M = camera_shift_matrix(W, H)
    f32 = dict(dtype=torch.float32, device=dev)
    plain = dict(trans=torch.empty((P, 4), **f32), final=torch.empty((P, 4), **f32), depth1=torch.empty(P, **f32))
    adapt = dict(final=torch.empty((P, 4), **f32))
    qt = None
    bal = None
    rp = None
    d_plain = ctx.make_resolve_desc(fb, BG, plain["trans"], plain["final"], plain["depth1"])
    stream = torch.cuda.current_stream()
    names = ["resolve", "quadtree", "balance", "adaptive", "reproject", "fallback"]

    def step(ev=None):
        nonlocal qt, bal, rp
        if ev: ev[0].record(stream)
        ctx.resolve_desc(d_plain)
        if ev: ev[1].record(stream)
        qt = ctx.quadtree(plain["final"], W, H, noit.QT_VARIANCE, 6, out=qt)
        if ev: ev[2].record(stream)
        bal = ctx.quadtree_balance(qt["tile_mask"], W, H, out=bal)
        if ev: ev[3].record(stream)
        ctx.resolve(fb, BG, want=(), out=adapt, half=hb, quarter=qb, cell_level=bal["cell_level"])
        if ev: ev[4].record(stream)
        rp = ctx.reproject(W, H, M, 1e-3, BG, plain["trans"], plain["depth1"], plain["depth1"], out=rp)
        if ev: ev[5].record(stream)
        ctx.resolve(fb, BG, want=(), out=dict(trans=rp["trans"], final=rp["final"], depth1=rp["depth"]),
                    pixel_list=rp["reject_list"], pixel_count=rp["reject_count"])
        if ev: ev[6].record(stream)

    # The same step with its two independent chains forked inside the graph: after the plain
    # resolve, frame 3 (reprojection + fallback, S8-S9) depends only on that resolve's outputs and
    # frame 2 (quadtree + balance + adaptive, S6-S7) only on its image, so the short launch-bound
    # quadtree kernels and the latency-bound fallback overlap with the other chain.  Chain B runs
    # on a side stream through a context of its own (a context's scratch -- tile counters -- is
    # stream-ordered, include/noit.h).
    ctx_b = noit.Noit(sc.weights, sc.mlp_precision)
    # the critical chain (frame 1 -> frame 2) is captured on a high-priority stream, frame 3 on a
    # default-priority one: where both have CTAs pending, the critical chain's go first
    side = torch.cuda.Stream(device=dev, priority=0)
    main_hp = torch.cuda.Stream(device=dev, priority=-1)

    def step_forked():
        nonlocal qt, bal, rp
        cur = torch.cuda.current_stream()
        ctx.resolve_desc(d_plain)
        side.wait_stream(cur)
        with torch.cuda.stream(side):
            rp = ctx_b.reproject(W, H, M, 1e-3, BG, plain["trans"], plain["depth1"], plain["depth1"], out=rp)
            ctx_b.resolve(fb, BG, want=(), out=dict(trans=rp["trans"], final=rp["final"], depth1=rp["depth"]),
                          pixel_list=rp["reject_list"], pixel_count=rp["reject_count"])
        qt = ctx.quadtree(plain["final"], W, H, noit.QT_VARIANCE, 6, out=qt)
        bal = ctx.quadtree_balance(qt["tile_mask"], W, H, out=bal)
        ctx.resolve(fb, BG, want=(), out=adapt, half=hb, quarter=qb, cell_level=bal["cell_level"])
        cur.wait_stream(side)

    # clocks are sampled from the warm-up to the end of the e2e leg (the timed region alone is a
    # few milliseconds: too short for nvidia-smi), i.e. always under this benchmark's load
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    for _ in range(max(args.warmup, 3)):
        step()
    torch.cuda.synchronize()
    events = [[torch.cuda.Event(enable_timing=True) for _ in range(7)] for _ in range(args.steps)]
    launches0 = ctx.launch_count
    if dist is not None:
        dist.barrier()
    torch.cuda.synchronize()
    for k in range(args.steps):
        step(events[k])
    torch.cuda.synchronize()
    if dist is not None:
        dist.barrier()
    launches = ctx.launch_count - launches0
    total_ms = events[0][0].elapsed_time(events[-1][6])
    total_ms = max_over_ranks(dist, total_ms, dev)
    eager_ms = total_ms
    # The step is launch-bound around its short kernels (seven launches + two memsets, ~15 us of
    # gaps): capture it once in a CUDA graph and time K replays -- that is the number `value`
    # reports; the eager pass above supplies the per-kernel times and the roofline.
    launch_mode = "eager"
    serial_graph_ms = None
    if not args.no_graph:
        def time_graph(fn):
            snap = (plain["final"].clone(), adapt["final"].clone(), rp["final"].clone(), rp["trans"].clone())
            graph = torch.cuda.CUDAGraph()
            with torch.cuda.graph(graph, stream=main_hp):
                fn()
            for _ in range(3):
                graph.replay()
            g0, g1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            if dist is not None:
                dist.barrier()
            torch.cuda.synchronize()
            cur = torch.cuda.current_stream()
            g0.record(cur)
            for _ in range(args.steps):
                graph.replay()
            g1.record(cur)
            torch.cuda.synchronize()
            if dist is not None:
                dist.barrier()
            # the replayed step did the same work: same frames, bit for bit
            now = (plain["final"], adapt["final"], rp["final"], rp["trans"])
            if not all(torch.equal(a, b) for a, b in zip(snap, now)):
                raise SystemExit("bench.py: graph replay produced different frames than the eager step")
            return max_over_ranks(dist, g0.elapsed_time(g1), dev)
        try:
            total_ms = time_graph(step)
            serial_graph_ms = total_ms
            launch_mode = "cuda graph replay of the whole step"
            if not args.no_fork:
                step_forked()                                      # eager once: nothing allocates under capture
                torch.cuda.synchronize()
                total_ms = time_graph(step_forked)
                launch_mode = ("cuda graph replay of the whole step, frame 3 (S8-S9) forked beside "
                               "frame 2 (S6-S7) after the plain resolve")
        except Exception as exc:                                   # capture refused: keep what was timed
            sys.stderr.write(f"bench.py: CUDA graph capture failed ({exc}); previous timing kept\n")
            torch.cuda.synchronize()
    per_kernel = {n: float(np.mean([e[i].elapsed_time(e[i + 1]) for e in events])) for i, n in enumerate(names)}
    resolve_ms = max_over_ranks(dist, per_kernel["resolve"], dev)

    # e2e: the same resolve through noit_resolve_host, pinned HOST buffers, copies inside the timing
    h_off = torch.from_numpy(fbh.offsets.view(np.int32)).pin_memory()
    h_depth = torch.from_numpy(fbh.depth).pin_memory()
    h_rgba = torch.from_numpy(fbh.rgba).pin_memory()
    h_final = torch.empty((P, 4), dtype=torch.float32).pin_memory()

    class HostFB:
        width, height, num_fragments, color_fmt = W, H, F, fb.color_fmt
        offsets, depth, rgba = h_off, h_depth, h_rgba

    e2e_steps = max(1, min(args.steps, 5))
    ctx.resolve_host(HostFB, BG, out_final=h_final)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    if dist is not None:
        dist.barrier()
    torch.cuda.synchronize()
    e0.record(stream)
    for _ in range(e2e_steps):
        ctx.resolve_host(HostFB, BG, out_final=h_final)
    e1.record(stream)
    torch.cuda.synchronize()
    e2e_ms = max_over_ranks(dist, e0.elapsed_time(e1) / e2e_steps, dev)
    # entry points outside the step (NEXT-2, NEXT-3): CUDA-event means, reported as `extras_ms`
    def timed(fn, n=20):
        for _ in range(3):
            fn()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(stream)
        for _ in range(n):
            fn()
        b.record(stream)
        torch.cuda.synchronize()
        return a.elapsed_time(b) / n
    tq = {"o": None}
    q16 = {"o": None}
    def run_temporal():
        tq["o"] = ctx.quadtree_temporal(plain["final"], W, H, qt["tile_mask"], out=tq["o"])
    def run_q16():
        q16["o"] = ctx.quadtree16(plain["final"], W, H, noit.QT_CORNER, 6, 0.02, out=q16["o"])
    # NEXT-4: inference cost of the 5-feature network vs the comparison system's 10-feature one
    # (same kernel shape; the paper reports a 35 % inference speed-up on RTX 5080)
    rng10 = np.random.default_rng(1)
    w931 = rng10.uniform(-0.2, 0.2, 931).astype(np.float32)
    x5 = torch.rand((P, 5), **f32)
    x10 = torch.rand((P, 10), **f32)
    y3 = torch.empty((P, 3), **f32)
    ctx32 = noit.Noit(sc.weights, noit.MLP_FP32)          # fp32 weights: the FFMA form of the network
    t5 = timed(lambda: ctx32.infer(x5, out=y3))
    t5m = timed(lambda: ctx.infer(x5, out=y3))             # bf16-rounded weights: tensor cores
    t10 = timed(lambda: ctx.infer_dfaoit(w931, x10, out=y3))
    extras = {"infer_5_features": t5, "infer_5_features_mma": t5m, "infer_10_features_dfaoit": t10,
              "inference_time_saved_by_5_features": 1.0 - t5 / t10,
              "quadtree_temporal": timed(run_temporal), "quadtree16_corner": timed(run_q16),
              "quadtree_balance": timed(lambda: ctx.quadtree_balance(qt["tile_mask"], W, H, out=bal))}
    # NEXT-4 (O12): the whole DFAOIT resolve (ten features built in the same scan, sigmoid network,
    # Eq. 3) against the 5-feature resolve with the same FFMA2 network form (fp32 weights) and
    # against the product path (bf16-rounded weights, tensor-core network): the resolve-level
    # counterpart of the paper's "10 -> 5 features: 35 % faster inference"
    outs10 = dict(trans=plain["trans"], final=plain["final"], depth1=plain["depth1"])
    t10r = timed(lambda: ctx.resolve_dfaoit(fb, w931, BG, want=(), out=outs10))
    t5f = timed(lambda: ctx32.resolve_desc(d_plain))
    t5m = timed(lambda: ctx.resolve_desc(d_plain))
    extras.update({"resolve_dfaoit_10_features_ffma2": t10r, "resolve_5_features_ffma2": t5f,
                   "resolve_5_features_mma": t5m, "resolve_time_saved_by_5_features_same_network_form": 1.0 - t5f / t10r,
                   "resolve_time_saved_by_5_features_product_path": 1.0 - t5m / t10r})
    # NEXT-4 (O8b): the step's reprojection with the bilinear fetch, into buffers of its own
    rpb = {"o": None}
    def run_rp(filt):
        rpb["o"] = ctx.reproject(W, H, M, 1e-3, BG, plain["trans"], plain["depth1"], plain["depth1"],
                                 out=rpb["o"], filter=filt)
    extras["reproject_nearest"] = timed(lambda: run_rp("nearest"))
    extras["reproject_bilinear"] = timed(lambda: run_rp("bilinear"))
    clocks = sampler.stop() if rank == 0 else None
    rejected = int(rp["reject_count"].item())
    hist = bal["hist"].cpu().numpy().view(np.uint32).tolist()
    scales = [float(v) for v in bal["scales"].cpu().numpy()]

    if rank == 0:
        peak, peak_src = peaks()
        ms_step = total_ms / args.steps
        # per-kernel algorithmic bytes of the step, this rank's frame or band
        lod_px = np.asarray([2, 1, 0, 0], np.int64)[
            bal["cell_level"].cpu().numpy().reshape((H + 7) // 8, (W + 7) // 8).repeat(8, 0).repeat(8, 1)[:H, :W]
        ].reshape(-1)
        rl = rp["reject_list"].cpu().numpy().view(np.uint32)[:rejected].astype(np.int64)
        F_rej = int(np.diff(fbh.offsets.astype(np.int64))[rl].sum())
        kb = step_bytes(fbh, sc.half, sc.quarter, lod_px, rejected, F_rej)
        kname = {"resolve": "resolve_staged_kernel<half,4,mma,ALL> (noit_resolve, S1-S5)",
                 "quadtree": "quadtree_kernel (noit_quadtree, S6)",
                 "balance": "balance_kernel (noit_quadtree_balance, NEXT-1)",
                 "adaptive": "coarse_g_kernel + resolve_staged_kernel<half,4,mma,ADAPTIVE> (noit_resolve, S7)",
                 "reproject": "reproject_kernel<nearest> (noit_reproject, S8)",
                 "fallback": "resolve_staged_kernel<half,2,ffma2,LIST> (noit_resolve, S9)"}
        roofline_all = [{"kernel": kname[k], "step": k, "bytes": int(kb[k]), "ms": per_kernel[k],
                         "achieved_gbs": kb[k] / (per_kernel[k] * 1e-3) / 1e9,
                         "frac": kb[k] / (per_kernel[k] * 1e-3) / 1e9 / peak} for k in names]
        rbytes = kb["resolve"]
        achieved = rbytes / (resolve_ms * 1e-3) / 1e9
        traffic, traffic_src = resolve_traffic()
        rec = {
            "metric": METRIC, "value": P_job / (resolve_ms * 1e-3) / 1e6, "unit": "Mpixels/s",
            "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": resolve_ms,
            "higher_is_better": True, "scaling": args.scaling if world > 1 else "weak", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic",
            "config": {"workload": WORKLOAD, "pixels": P_job, "fragments": F_job,
                       "what_is_timed": WHAT_IS_TIMED, "l2": L2_NOTE,
                       "sharding": ("none" if world == 1 else
                                    ("one frame in fragment-balanced 64-row bands, no collective" if args.scaling == "strong"
                                     else "one frame per rank (seed = rank), no collective"))},
            "timing": "CUDA events on the launching stream around noit_resolve, inside the whole-path step loop",
            "fragments_per_s": F_job / (resolve_ms * 1e-3),
            "resolve_mpix_s": P_job / (resolve_ms * 1e-3) / 1e6,
            "resolve_gfrag_s": F_job / (resolve_ms * 1e-3) / 1e9,
            "kernel_ms": per_kernel,
            "step_frames": 3, "step_launch": launch_mode, "step_ms": ms_step,
            "step_mpix_s": 3 * P_job / (ms_step * 1e-3) / 1e6,
            "step_ms_eager": eager_ms / args.steps,
            "step_ms_serial_graph": None if serial_graph_ms is None else serial_graph_ms / args.steps,
            "extras_ms": extras,
            "roofline": {"bound": "hbm", "kernel": kname["resolve"], "achieved": achieved,
                         "peak": peak, "unit": "GB/s", "frac": achieved / peak, "peak_source": peak_src,
                         "algorithmic_bytes": rbytes, "bytes_formula": "4(P+1) + 12F + 2*16P + 4P",
                         "traffic": traffic, "traffic_source": traffic_src},
            "roofline_all": roofline_all,
            "e2e": {"value": P_job / (e2e_ms * 1e-3) / 1e6, "unit": "Mpixels/s",
                    "what": "noit_resolve_host on the same frame, pinned host buffers",
                    "h2d_bytes_per_step": 4 * (P + 1) + 12 * F, "d2h_bytes_per_step": 16 * P,
                    "ms_per_step": e2e_ms},
            "gpu_launches": launches, "clocks": clocks,
            "tile_hist": hist, "demand_index_and_scales": scales, "rejected_fraction": rejected / P,
        }
        if world == 1 and not args.no_cpu_baseline:
            rec["cpu_baseline"] = cpu_baseline(sc)
        print(json.dumps(rec))
    if dist is not None:
        dist.destroy_process_group()


def cpu_baseline(sc) -> dict:
    """The oracle as it stands on this box's host cores: plain resolve of the same frame,
    repeated for about 10 s (bounded), same metric as `resolve_mpix_s`."""
    import oracle
    w_eff = oracle.effective_weights(sc.weights, sc.mlp_precision)
    oracle.resolve(sc.full, w_eff, BG)
    n, t0 = 0, time.perf_counter()
    while n < 3 or (time.perf_counter() - t0 < 10.0 and n < 200):
        oracle.resolve(sc.full, w_eff, BG)
        n += 1
    dt = (time.perf_counter() - t0) / n
    return {"value": sc.full.num_pixels / dt / 1e6, "unit": "Mpixels/s", "cores": oracle.num_threads(),
            "kind": "oracle", "ms_per_frame": dt * 1e3,
            "sample": f"plain resolve (S1-S5) of the whole cfg3 frame, {n} repetitions"}


def run_info(args):
    """`--config cfgK` (information only, not the contract line): the plain resolve -- and for cfg4
    the quadtree + balance + adaptive resolve -- of BASELINE.json's other configs, CUDA-event means
    with an L2 flush (a 512 MB fill) between iterations where the inputs fit L2."""
    import torch

    import noit_scenes
    import paper_2606_16747_b200 as noit
    torch.cuda.set_device(0)
    dev = torch.device("cuda", 0)
    name = args.config
    if name.startswith("synth:"):
        return run_synth(args, name)
    if name not in ("cfg1", "cfg2", "cfg3", "cfg4", "cfg5"):
        raise SystemExit(f"bench.py: unknown --config {name}")
    if name == "cfg5":
        seq = noit_scenes.cfg5(0)
        sc = noit_scenes.Scene("cfg5-frame0", seq.frame(0), weights=seq.weights, mlp_precision=seq.mlp_precision)
    else:
        sc = {"cfg1": noit_scenes.cfg1, "cfg2": noit_scenes.cfg2, "cfg3": noit_scenes.cfg3,
              "cfg4": noit_scenes.cfg4}[name](0)
    fbh = sc.full
    P, F = fbh.num_pixels, fbh.num_fragments
    cb = fbh.rgba.dtype.itemsize * 4
    fb = noit.DeviceFragBuf.from_host(fbh, dev)
    ctx = noit.Noit(sc.weights, sc.mlp_precision)
    f32 = dict(dtype=torch.float32, device=dev)
    out = dict(trans=torch.empty((P, 4), **f32), final=torch.empty((P, 4), **f32), depth1=torch.empty(P, **f32))
    d_plain = ctx.make_resolve_desc(fb, BG, out["trans"], out["final"], out["depth1"])
    flush = torch.empty(512 << 20, dtype=torch.uint8, device=dev)
    stream = torch.cuda.current_stream()

    def timed(fn, n):
        for _ in range(3):
            fn()
        ms = []
        for _ in range(n):
            flush.fill_(1)
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(stream)
            fn()
            b.record(stream)
            torch.cuda.synchronize()
            ms.append(a.elapsed_time(b))
        return float(np.mean(ms))

    peak, peak_src = peaks()
    rec = {"info": True, "config": name, "pixels": P, "fragments": F, "steps": args.steps,
           "l2": "512 MB fill between iterations"}
    t = timed(lambda: ctx.resolve_desc(d_plain), args.steps)
    rbytes = resolve_bytes(P, F, cb, 2, True)
    rec.update(resolve_ms=t, resolve_mpix_s=P / t / 1e3, resolve_gfrag_s=F / t / 1e6,
               resolve_gbs=rbytes / t / 1e6, resolve_frac_of_hbm_peak=rbytes / t / 1e6 / peak,
               mlp_us_at_fp32_peak=P * 1440 / 74.4e12 * 1e6, peak_source=peak_src)
    if sc.half is not None:
        hb, qb = (noit.DeviceFragBuf.from_host(b, dev) for b in (sc.half, sc.quarter))
        W, H = fbh.width, fbh.height
        qt = ctx.quadtree(out["final"], W, H, noit.QT_VARIANCE, 6)
        bal = ctx.quadtree_balance(qt["tile_mask"], W, H)
        adapt = dict(final=torch.empty((P, 4), **f32))
        ta = timed(lambda: ctx.resolve(fb, BG, want=(), out=adapt, half=hb, quarter=qb,
                                       cell_level=bal["cell_level"]), args.steps)
        # the paper's frame-global control with pass 2 at half and pass 3 at quarter resolution
        forced = torch.tensor([2.0, 0.5, 0.25], **f32)
        tg = timed(lambda: ctx.resolve(fb, BG, want=(), out=adapt, half=hb, quarter=qb, pass_scales=forced),
                   args.steps)
        rec.update(global_half_quarter_ms=tg, global_speedup_over_plain=t / tg)
        lv = bal["cell_level"].cpu().numpy()
        rec.update(adaptive_ms=ta, adaptive_speedup_over_plain=t / ta,
                   tile_hist=bal["hist"].cpu().numpy().view(np.uint32).tolist(),
                   cell_fraction_per_level=[float((lv == k).mean()) for k in range(4)],
                   scales=[float(v) for v in bal["scales"].cpu().numpy()])
    print(json.dumps(rec))


def run_synth(args, name):
    """`--config synth:LO-HI`: a 1920x1080 frame whose every pixel holds U{LO..HI} fragments (random
    depths and fp16 colours drawn on the device): separates the per-pixel cost of the resolve from
    its per-fragment cost (profiles/r02_resolve.md)."""
    import torch

    import noit_scenes
    import paper_2606_16747_b200 as noit
    lo, hi = (int(v) for v in name.split(":")[1].split("-"))
    torch.cuda.set_device(0)
    dev = torch.device("cuda", 0)
    W, H = 1920, 1080
    P = W * H
    counts = np.random.default_rng(1).integers(lo, hi + 1, P)
    off = np.zeros(P + 1, np.uint32)
    off[1:] = np.cumsum(counts)
    F = int(off[-1])
    torch.manual_seed(1)
    fb = noit.DeviceFragBuf(W, H, torch.from_numpy(off.view(np.int32)).to(dev),
                            torch.rand(F, device=dev) * 0.98 + 0.01, torch.rand((F, 4), device=dev).half())
    ctx = noit.Noit(noit_scenes.mlp_weights(0), noit.MLP_BF16)
    f32 = dict(dtype=torch.float32, device=dev)
    out = dict(trans=torch.empty((P, 4), **f32), final=torch.empty((P, 4), **f32), depth1=torch.empty(P, **f32))
    d = ctx.make_resolve_desc(fb, BG, out["trans"], out["final"], out["depth1"])
    flush = torch.empty(512 << 20, dtype=torch.uint8, device=dev)
    stream = torch.cuda.current_stream()
    for _ in range(3):
        ctx.resolve_desc(d)
    ms = []
    for _ in range(args.steps):
        flush.fill_(1)
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(stream)
        ctx.resolve_desc(d)
        b.record(stream)
        torch.cuda.synchronize()
        ms.append(a.elapsed_time(b))
    t = float(np.mean(ms))
    peak, peak_src = peaks()
    rbytes = resolve_bytes(P, F, 8, 2, True)
    print(json.dumps({"info": True, "config": name, "pixels": P, "fragments": F, "fragments_per_tile": F / (P / 32),
                      "steps": args.steps, "resolve_ms": t, "resolve_gbs": rbytes / t / 1e6,
                      "resolve_frac_of_hbm_peak": rbytes / t / 1e6 / peak, "peak_source": peak_src,
                      "memory_floor_ms": rbytes / peak / 1e6}))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--scaling", default="weak", choices=["weak", "strong"],
                    help="N > 1: one frame per rank (weak) or one frame split into row bands (strong)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-graph", action="store_true", help="time the step eagerly (no CUDA graph)")
    ap.add_argument("--no-fork", action="store_true", help="graph replay of the serial step only")
    ap.add_argument("--config", default=None,
                    help="information only: time the plain resolve of one of BASELINE.json's other configs "
                         "(cfg1 .. cfg5), or of a synthetic 1080p frame with lo..hi fragments in every pixel "
                         "(synth:LO-HI): the rate each path of the kernel reaches")
    args = ap.parse_args()
    if os.environ.get("NOIT_BENCH_DRYRUN"):
        return run_dryrun(args)
    if args.impl == "reference":
        return run_reference(args)
    if args.config:
        return run_info(args)
    return run_ours(args)


if __name__ == "__main__":
    main()
