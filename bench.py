#!/usr/bin/env python
"""bench.py - whole-hot-path benchmark of libvr on B200 (contract: see DESIGN.md "Measurement").

A step = one frame of the workload's camera orbit through every row of SURVEY.md 8(a):
S1 vr_set_view + vr_sort_bricks (host), S2-S4 vr_render_bricks (the ray marcher, per-brick partial
images), S5 vr_composite_bricks (sort-last fold), S6 the tiled frame when the workload has panels.
The cube (S0) is generated on the device once, before the timed region.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload C3] [--impl reference]

N > 1 (torchrun): "replicas only" - every rank holds its own copy of the cube and renders its own
frames of the orbit; there is no data-path collective (BASELINE.json north_star: "no sharding and
no collectives").  `--impl reference` times the CPU oracle (oracle/), as it stands, on a bounded
pixel sample of the same workload.
"""
from __future__ import annotations

import argparse
import json
import math
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_1012_2909_b200 import workloads as wl  # noqa: E402
from paper_1012_2909_b200.replicas import orbit_frame as _orbit_frame, reduce_run  # noqa: E402

METRIC = "ray samples/s (nominal lattice samples inside the cube; BASELINE.json metric)"


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            return json.load(f), "measured (MEASURED_PEAKS.json)"
    return {"hbm_gbs": 6650.0}, "fallback (B200_PROFILING.md: 6.65 TB/s)"


class ClockSampler(threading.Thread):
    """Samples SM clocks and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.stop_flag, self.samples, self.reasons, self.max_mhz = index, False, [], set(), None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
        except Exception:
            self.nv = None

    def run(self):
        if self.nv is None:
            return
        nv = self.nv
        names = {
            getattr(nv, "nvmlClocksEventReasonHwSlowdown", 0x8): "hw_slowdown",
            getattr(nv, "nvmlClocksEventReasonHwThermalSlowdown", 0x40): "hw_thermal_slowdown",
            getattr(nv, "nvmlClocksEventReasonSwThermalSlowdown", 0x20): "sw_thermal_slowdown",
            getattr(nv, "nvmlClocksEventReasonSwPowerCap", 0x4): "sw_power_cap",
        }
        while not self.stop_flag:
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                try:
                    r = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                except Exception:
                    r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for bit, name in names.items():
                    if r & bit:
                        self.reasons.add(name)
            except Exception:
                pass
            time.sleep(0.05)

    def result(self):
        self.stop_flag = True
        if self.nv is None or not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": ["unavailable"]}
        return {"sm_mhz": float(np.median(self.samples)), "sm_max_mhz": float(self.max_mhz),
                "reasons": sorted(self.reasons), "samples": len(self.samples)}


def orbit_frame(w, step_index, n_steps, rank, world):
    """Frame index of the 360-frame orbit rendered at a given step (paper_1012_2909_b200/replicas.py)."""
    return _orbit_frame(step_index, n_steps, rank, world)


# dram__bytes_read.sum + dram__bytes_write.sum per launch of the marcher, from the committed
# `ncu --set full` captures (profiles/r1d_c3_render_occ_full.md: orbit frames 0 and 180, 11.26 and 8.08 GB read + written, their mean; r1d_c3_mip_render_ls_full.md: frame 0).  None: not captured.
NCU_TRAFFIC_BYTES = {("C3", "ea"): 9.67e9, ("C3", "mip"): 70.3e9}
# smsp__inst_executed.sum (warp instructions) per launch from the same captures, and the issue peak
# DESIGN.md section 8 derives: 148 SMs x 4 schedulers x 1 warp instruction per clock.
NCU_WARP_INSTRUCTIONS = {("C3", "ea"): 4.54e9, ("C3", "mip"): 8.28e9}
ISSUE_SLOTS_PER_CLOCK = 148 * 4

MARCHER = {(0, 0): "render_tiles_kernel<EA> (ray per thread)", (0, 1): "render_tiles_kernel<EA> (ray per thread)",
           (0, 2): "render_tiles_kernel<EA> (ray per thread, macro-cell runs)",
           (0, 3): "render_tiles_kernel<EA> (ray per thread, macro-cell runs + occupancy bits)",
           (3, 3): "render_occ_kernel (lockstep: occupancy test, compaction, cp.async gather, fold)"}


class Job:
    """One rank's resident cube + context."""

    def __init__(self, w, device, mode="ea", shard=None, dist=None):
        import torch
        from paper_1012_2909_b200 import vr
        self.torch, self.vr, self.w = torch, vr, w
        self.mode = vr.MODE_EA if mode == "ea" else vr.MODE_MIP
        self.px_bytes = 16 if mode == "ea" else 4
        torch.cuda.set_device(device)
        self.ctx = vr.Context(device)
        self.shard, self.dist = None, dist
        if shard is not None:                     # (rank, world): this rank holds one z-slab of the bricks
            from paper_1012_2909_b200 import sortlast
            self.sortlast = sortlast
            self.shard = sortlast.Shard(self.ctx, w.dims, w.brick, shard[0], shard[1])
            self.shard.bind()
            cb, mb = self.shard.layout()
        else:
            cb, mb = vr.cube_layout(w.dims, w.brick)
        self.d_cube = torch.empty(max(cb // 4, 1), dtype=torch.float32, device="cuda")
        self.d_meta = torch.empty(max(mb, 1), dtype=torch.uint8, device="cuda")
        t0 = time.perf_counter()
        self.ctx.generate_cube(w.seed, w.dims, w.brick, self.d_cube, self.d_meta, sources=wl.make_sources(w),
                               zero_boxes=wl.make_zero_boxes(w), continuum=w.continuum)
        torch.cuda.synchronize()
        self.gen_seconds = time.perf_counter() - t0
        self.tf = wl.TFS[w.tf]()
        self.ctx.set_transfer_function(*self.tf)
        self.W, self.H = w.frame
        self.cols, self.rows = w.panels
        self.pw, self.ph = self.W // self.cols, self.H // self.rows
        ch = 4 if mode == "ea" else 1
        self.frame = torch.zeros((self.H, self.W, ch), dtype=torch.float32, device="cuda")
        self.arena = None
        self.h_frame = torch.empty((self.H, self.W, ch), dtype=torch.float32).pin_memory()
        self.step_events = []
        self.bg = (0.0, 0.0, 0.0, 0.0)
        self.march_events = []
        self.alg_bytes = 0

    def _arena(self, nbytes):
        if self.arena is None or self.arena.numel() < nbytes:
            self.arena = self.torch.empty(int(nbytes * 1.25) + 256, dtype=self.torch.uint8, device="cuda")
        return self.arena

    def step(self, frame_index, timed_events=False, set_tf=False):
        """S1 + S2-S5 (+ S6) for one frame, sort-last path."""
        w, vr, ctx, torch = self.w, self.vr, self.ctx, self.torch
        M = wl.config_camera(w, frame_index)
        if set_tf:
            ctx.set_transfer_function(*self.tf)
        brick_vox = 1
        for b, n in zip(w.brick, w.dims):
            brick_vox *= min(b, n)
        if self.shard is not None:
            # sharded sort-last (paper_1012_2909_b200/sortlast.py): own bricks -> one partial frame, strips
            # exchanged, folded in the slabs' visibility order, gathered
            sh, sl = self.shard, self.sortlast
            ctx.set_view(M, self.W, self.H, w.step)
            if timed_events:
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record()
            part = sh.render_partial(torch, self.mode, self.W, self.H, w.tau)
            if timed_events:
                e1.record()
                self.march_events.append((e0, e1))
                self.alg_bytes += 4 * brick_vox * (sh.end - sh.first) + self.H * self.W * self.px_bytes
            if getattr(self, "slab_only", False):
                self.frame = part
            else:
                versions = sl.exchange_strips(self.dist, part, sh.world)
                strip = sh.fold_strip(torch, self.mode, versions, self.W, self.H, self.bg)
                self.frame = sl.gather_strips(self.dist, strip, sh.world, self.H)
            if timed_events:
                e = torch.cuda.Event(enable_timing=True)
                e.record()
                self.step_events.append(e)
            return
        for r in range(self.rows):
            for c in range(self.cols):
                Mp = M if (self.cols, self.rows) == (1, 1) else wl.panel_matrix(M, self.cols, self.rows, c, r)
                ctx.set_view(Mp, self.pw, self.ph, w.step)
                ctx.set_viewport(c * self.pw, r * self.ph, self.W)
                ids = ctx.sort_bricks(self.mode)
                parts, n, nbytes = ctx.partial_layout(self.mode, ids)
                vr.Context.bind_partials(parts, n, self._arena(nbytes))
                if timed_events:
                    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                    e0.record()
                ctx.render_bricks(self.mode, parts, n, w.tau)
                if timed_events:
                    e1.record()
                    self.march_events.append((e0, e1))
                    # algorithmic bytes of this launch: the active in-frustum bricks
                    # read once + the partial images written once
                    self.alg_bytes += 4 * brick_vox * n + nbytes          # nbytes: the partial images (16 or 4 B per pixel)
                ctx.composite_bricks(self.mode, parts, n, self.frame, self.bg)
        if timed_events:
            e = torch.cuda.Event(enable_timing=True)
            e.record()
            self.step_events.append(e)


def oracle_sample(job, frame_index, tile, precision_name="F64"):
    """Time the oracle, as it stands, on a tile x tile pixel block at the frame centre of the
    same frame (sort-last semantics, same partition, same tau).  Returns (seconds, counters)."""
    from oracle import ovr
    w, torch = job.w, job.torch
    M = wl.config_camera(w, frame_index)
    cx, cy = job.W // 2, job.H // 2
    xs = np.arange(cx - tile // 2, cx - tile // 2 + tile)
    ys = np.arange(cy - tile // 2, cy - tile // 2 + tile)
    pix = np.stack(np.meshgrid(xs, ys), axis=-1).reshape(-1, 2).astype(np.int32)
    brick = tuple(min(b, n) for b, n in zip(w.brick, w.dims))
    touched = ovr.bricks_touched(M, job.W, job.H, w.step, w.dims, brick, pix)
    bricks = {}
    g = [-(-n // b) for n, b in zip(w.dims, brick)]
    for b in touched:                       # fetch the cube bytes back from the device (untimed)
        bi = (b % g[0], (b // g[0]) % g[1], b // (g[0] * g[1]))
        ext = [min(bb, n - i * bb) for i, bb, n in zip(bi, brick, w.dims)]
        t = torch.empty(ext[0] * ext[1] * ext[2], dtype=torch.float32, device="cuda")
        job.ctx.download_brick(int(b), t)
        bricks[int(b)] = t.cpu().numpy()
    torch.cuda.synchronize()
    vol = ovr.Volume(w.dims, brick, bricks)
    t0 = time.perf_counter()
    omode = ovr.EA if job.mode == job.vr.MODE_EA else ovr.MIP
    _, _, cnt = ovr.render(vol, M, job.W, job.H, w.step, omode, getattr(ovr, precision_name), tf=job.tf,
                           split=ovr.SPLIT_SORTLAST, partition=brick, tau=w.tau, bg=job.bg, pixels=pix)
    return time.perf_counter() - t0, cnt, len(touched)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=24)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="C3", choices=sorted(wl.CONFIGS))
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--mode", default="ea", choices=["ea", "mip"], help="emission-absorption (default) or MIP")
    ap.add_argument("--sharded", action="store_true",
                    help="N ranks share ONE cube: bricks sharded in z-slabs, sort-last exchange over NCCL (NEXT-1, "
                         "strong scaling); default: N independent replicas")
    ap.add_argument("--slab", default=None, metavar="R/W",
                    help="render only slab R of a W-way split of the bricks (what rank R of --sharded would render; no "
                         "exchange): the per-rank cost of NEXT-1 measured on one GPU")
    ap.add_argument("--next-rows", action="store_true",
                    help="time the catalogue overlay and the output pyramid (SURVEY.md 8(f) 2 and 3) instead of the marcher")
    ap.add_argument("--frame", default=None, help="WxH: render one frame of this size instead of the workload's "
                                                   "(BASELINE.json configs[4]: C5's 1920x1080 MIP)")
    ap.add_argument("--cpu-seconds", type=float, default=15.0, help="target CPU time of the oracle sample")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "b200" else args.warmup

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if args.impl == "reference" and rank != 0:
        return 0

    import torch
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the hot path has no CPU fallback")
    dist = None
    if world > 1 and args.impl == "b200":
        import torch.distributed as dist
        torch.cuda.set_device(local_rank)
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    w = wl.CONFIGS[args.workload]
    if args.frame:
        from dataclasses import replace
        w = replace(w, frame=tuple(int(v) for v in args.frame.lower().split("x")), panels=(1, 1))
    if args.next_rows:
        return run_next_rows(args)
    slab = None
    if args.slab:
        slab = tuple(int(v) for v in args.slab.split("/"))
        if world != 1 or args.sharded or not (0 <= slab[0] < slab[1]):
            raise SystemExit("--slab R/W runs on one GPU, without --sharded")
    if (args.sharded or slab) and w.panels != (1, 1):
        raise SystemExit("--sharded renders single-panel frames (use --frame WxH for the tiled workloads)")
    job = Job(w, local_rank, args.mode, shard=slab if slab else ((rank, world) if args.sharded else None), dist=dist)
    job.slab_only = slab is not None
    frank, fworld = (0, 1) if args.sharded else (rank, world)          # sharded: every rank renders every frame
    vr = job.vr
    config = {"workload": f"{w.name}: {w.dims[0]}x{w.dims[1]}x{w.dims[2]} float32 cube, {w.brick[0]}^3 bricks, "
                          f"{w.frame[0]}x{w.frame[1]} frame ({w.panels[0]}x{w.panels[1]} panels), step {w.step}, "
                          f"{'EA tf-' + w.tf + ' tau=' + str(w.tau) if args.mode == 'ea' else 'MIP'}, sort-last path, orbit frames spread over 360 deg",
              "cube_gib": round(w.n_voxels * 4 / 2 ** 30, 3), "n_sources": w.n_sources,
              "l2_policy": "inputs larger than L2 (cube >> 126 MB); no explicit flush",
              "e2e_policy": "matrix + table host->device and frame device->pinned host every step; two frame buffers, frame "
                            "i's copy overlaps frame i+1's render, the host waits for frame i-1 before issuing frame i+1",
              "replicas": 1 if args.sharded else world, "shards": world if args.sharded else 1, "slab": args.slab,
              "generate_seconds": round(job.gen_seconds, 3)}

    if args.impl == "reference":
        return run_reference(args, job, config)

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    for i in range(args.warmup):
        job.step(orbit_frame(w, i, args.steps, frank, fworld))
    job.ctx.reset_counters()
    sampler = ClockSampler(local_rank)
    barrier()
    sampler.start()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev0.record()
    for i in range(args.steps):
        job.step(orbit_frame(w, i, args.steps, frank, fworld), timed_events=True)
    ev1.record()
    barrier()
    clocks = sampler.result()
    ms_total = ev0.elapsed_time(ev1)
    marks = [ev0] + job.step_events
    frame_ms = sorted(a.elapsed_time(b) for a, b in zip(marks, marks[1:]))
    cnt = job.ctx.get_counters()
    march_ms = sum(a.elapsed_time(b) for a, b in job.march_events)
    n_march = len(job.march_events)

    ms_total, (nominal, taken, launches) = reduce_run(
        dist, "cuda", ms_total, [cnt["nominal_samples"], cnt["taken_samples"], cnt["kernel_launches"]])

    # ---- e2e: the same step through the public API with HOST buffers in the timed region: the
    # view matrix and the transfer-function table go host -> device every step (as kernel
    # parameters / table upload), the finished frame comes back device -> pinned host memory.
    job.ctx.reset_counters()
    barrier()
    # Two frame buffers: frame i's device -> host copy runs on a copy stream while frame i + 1 is rendered;
    # the host takes delivery of frame i - 1 (waits for its copy) before it issues frame i + 1.
    frames = [job.frame, torch.zeros_like(job.frame)]
    h_frames = [job.h_frame, torch.empty_like(job.h_frame).pin_memory()]
    copy_stream = torch.cuda.Stream()
    copied = [None, None]
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for i in range(args.steps):
        b = i % 2
        if copied[b] is not None:
            torch.cuda.current_stream().wait_event(copied[b])      # the buffer's previous frame has left the device
        job.frame = frames[b]
        job.step(orbit_frame(w, i, args.steps, frank, fworld), set_tf=True)
        src = job.frame                                             # (the sharded path returns a new tensor)
        rendered = torch.cuda.Event()
        rendered.record()
        with torch.cuda.stream(copy_stream):
            copy_stream.wait_event(rendered)
            h_frames[b].copy_(src, non_blocking=True)
            src.record_stream(copy_stream)
            copied[b] = torch.cuda.Event()
            copied[b].record()
        if i > 0:
            copied[1 - b].synchronize()                             # frame i - 1 is in host memory
    copied[(args.steps - 1) % 2].synchronize()
    torch.cuda.synchronize()
    e2e_s = time.perf_counter() - t0
    job.frame = frames[0]
    cnt2 = job.ctx.get_counters()
    e2e_s, (e2e_nominal,) = reduce_run(dist, "cuda", e2e_s, [cnt2["nominal_samples"]])

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return 0

    peaks, peak_src = measured_peaks()
    peak = float(peaks["hbm_gbs"])
    plan = job.ctx.get_plan(job.mode)
    kernel = MARCHER.get((plan["variant"], plan["skip_level"]),
                         "render_ls_kernel<EA> (lockstep, cp.async gather)" if plan["variant"] == 3 else "render_tiles_kernel<EA>")
    if args.mode == "mip":
        kernel = ("render_ls_kernel<MIP> (lockstep, cp.async gather, warp-reduced maximum)" if plan["variant"] == 3
                  else "render_tiles_kernel<MIP> (ray per thread)")
    traffic = NCU_TRAFFIC_BYTES.get((w.name, args.mode)) if not args.frame else None
    launch_s = march_ms / max(n_march, 1) * 1e-3
    winst = NCU_WARP_INSTRUCTIONS.get((w.name, args.mode)) if not args.frame else None
    issue = None
    if winst and launch_s > 0 and clocks.get("sm_mhz"):
        ipeak = ISSUE_SLOTS_PER_CLOCK * clocks["sm_mhz"] * 1e6 / 1e9
        issue = {"bound": "alu", "achieved": winst / launch_s / 1e9, "peak": ipeak, "unit": "G warp-instructions/s",
                 "frac": winst / launch_s / 1e9 / ipeak,
                 "note": "warp instructions per launch from the committed ncu capture / live launch time; peak = 148 SMs x 4 "
                         "schedulers x the SM clock sampled during the run: what actually bounds the occupancy marcher"}
    achieved = (job.alg_bytes / max(n_march, 1)) / (march_ms / max(n_march, 1) * 1e-3) / 1e9 if march_ms > 0 else 0.0
    cpu = None
    if world == 1 and not slab:           # a slab holds only its own bricks: no oracle sample
        tile = 8
        sec, c, nb = oracle_sample(job, orbit_frame(w, 0, args.steps, 0, 1), tile)
        if c["nominal"] > 0 and sec > 0:
            scale = args.cpu_seconds / max(sec, 1e-3)
            tile2 = int(min(256, max(8, tile * math.sqrt(scale))))
            if tile2 > tile:
                sec, c, nb = oracle_sample(job, orbit_frame(w, 0, args.steps, 0, 1), tile2)
                tile = tile2
        cpu = {"value": c["nominal"] / sec if sec > 0 else 0.0, "unit": "samples/s", "cores": 1, "kind": "oracle",
               "sample": f"fp64 oracle, sort-last, the {tile}x{tile}-pixel block at the centre of orbit frame 0 "
                         f"({c['nominal']} nominal samples, {nb} bricks fetched back from the device, {sec:.2f} s)"}

    out = {
        "metric": METRIC, "value": nominal / (ms_total * 1e-3), "unit": "samples/s",
        "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_total / args.steps, "frames_per_s": args.steps * fworld / (ms_total * 1e-3),
        "frame_ms": {"median": frame_ms[len(frame_ms) // 2], "p95": frame_ms[min(len(frame_ms) - 1, int(0.95 * len(frame_ms)))],
                     "min": frame_ms[0], "max": frame_ms[-1], "note": "rank 0, device time between consecutive frames of the orbit"},
        "higher_is_better": True, "scaling": "strong" if args.sharded else "weak", "vs_baseline": None, "dtype": "f32",
        "data": "synthetic", "config": config,
        "nominal_samples_per_step": nominal / (args.steps * fworld),
        "taken_samples_per_s": taken / (ms_total * 1e-3),
        "gpu_launches": launches,
        "clocks": clocks,
        "e2e": {"value": e2e_nominal / e2e_s, "unit": "samples/s", "ms_per_step": e2e_s * 1e3 / args.steps,
                "h2d_bytes_per_step": (64 + 4096 + 8) * job.cols * job.rows,
                "d2h_bytes_per_step": job.H * job.W * job.px_bytes},
        "roofline": {"bound": "hbm", "kernel": kernel, "achieved": achieved, "peak": peak,
                     "unit": "GB/s", "frac": achieved / peak if peak else None, "traffic": traffic,
                     "peak_source": peak_src, "launch_ms": march_ms / max(n_march, 1),
                     "share_of_step": march_ms / ms_total if ms_total else None,
                     "algorithmic_bytes_per_launch": job.alg_bytes / max(n_march, 1),
                     "dram_gbs_from_traffic": traffic / launch_s / 1e9 if traffic and launch_s > 0 else None,
                     "issue": issue,
                     "plan": plan,
                     "note": "algorithmic bytes = 4 B x voxels of the active in-frustum bricks at the configured brick "
                             "size + partial images (SURVEY.md 8(d)); skipping below the brick level (macro-cells, "
                             "occupancy bits) reads fewer bytes than that, so frac can exceed 1: `traffic` is what "
                             "the launch really moved"},
        "cpu_baseline": cpu,
    }
    print(json.dumps(out))
    if dist is not None:
        dist.destroy_process_group()
    return 0


def run_next_rows(args):
    """Timings of vr_overlay_catalogue and vr_build_pyramid (CUDA events, inputs resident in HBM)."""
    import torch
    from paper_1012_2909_b200 import vr
    ctx = vr.Context(0)

    def timeit(fn, n=10):
        fn()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(n):
            fn()
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / n

    out = {"impl": "b200", "what": "NEXT rows: catalogue overlay and output pyramid", "overlay": [], "pyramid": None}
    W, H = 1920, 1080
    for name in ("C3", "C5"):
        w = wl.CONFIGS[name]
        src = wl.make_sources(w)
        boxes = torch.from_numpy(src[:, wl.S_XLO:wl.S_ZHI + 1].astype(np.int32)).cuda()
        col = torch.rand((boxes.shape[0], 4), device="cuda")
        ctx.set_view(wl.perspective_camera(w.dims, (W, H), azimuth_deg=30.0), W, H, 0.5)
        frame = torch.zeros((H, W, 4), device="cuda")
        pick = torch.zeros((H, W), dtype=torch.int32, device="cuda")
        ms = timeit(lambda: ctx.overlay_catalogue(boxes, col, None, frame, pick))
        out["overlay"].append({"catalogue": f"{name}: {boxes.shape[0]} source boxes", "frame": f"{W}x{H}", "ms": ms,
                               "covered_pixels": int((pick > 0).sum().item())})
    Wp, Hp = 9600, 5400
    frame = torch.rand((Hp, Wp, 4), device="cuda")
    levels, nbytes = vr.pyramid_layout(Wp, Hp, 256)
    buf = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
    ms = timeit(lambda: ctx.build_pyramid(frame, Wp, Hp, Wp, buf, 256))
    out["pyramid"] = {"frame": f"{Wp}x{Hp}", "tile": 256, "levels": len(levels), "bytes_out": nbytes, "ms": ms}
    print(json.dumps(out))
    return 0


def run_reference(args, job, config):
    """The reference arm of this tier = the oracle, timed as it stands on the host cores."""
    w = job.w
    budget = 150.0 / max(1, args.steps + args.warmup)
    tile = 8
    sec, c, nb = oracle_sample(job, 0, tile)
    if sec > 0:
        tile = int(min(128, max(4, tile * math.sqrt(budget / max(sec, 1e-3)))))
    for i in range(args.warmup):
        oracle_sample(job, orbit_frame(w, i, args.steps, 0, 1), tile)
    total_s, total_n = 0.0, 0
    for i in range(args.steps):
        sec, c, nb = oracle_sample(job, orbit_frame(w, i, args.steps, 0, 1), tile)
        total_s += sec
        total_n += c["nominal"]
    value = total_n / total_s if total_s > 0 else 0.0
    out = {"impl": "reference", "metric": METRIC, "value": value, "unit": "samples/s", "n_gpus": args.gpus,
           "steps": args.steps, "warmup": args.warmup, "ms_per_step": total_s * 1e3 / max(1, args.steps),
           "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
           "config": config,
           "cpu_baseline": {"value": value, "unit": "samples/s", "cores": 1, "kind": "oracle",
                            "sample": f"fp64 oracle, sort-last, a {tile}x{tile}-pixel block at the frame centre per step"},
           "e2e": {"value": value, "unit": "samples/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(out))
    return 0


if __name__ == "__main__":
    sys.exit(main())
