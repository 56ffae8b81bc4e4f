#!/usr/bin/env python
"""bench.py - whole-hot-path benchmark of libvr on B200 (contract: see DESIGN.md "Measurement").

A step = one frame of the workload's camera orbit through every row of SURVEY.md 8(a):
S1 vr_set_view + vr_sort_bricks (host), S2-S4 vr_render_bricks (the ray marcher, per-brick partial
images), S5 vr_composite_bricks (sort-last fold), S6 the tiled frame when the workload has panels.
The cube (S0) is generated on the device once, before the timed region.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload C3] [--mode ea|mip] [--impl reference]

The headline line is C3 (BASELINE.json configs[2]: the 64 GiB cube at 1920 x 1080, emission-
absorption).  With the default arguments on one GPU the same JSON line also carries `configs`: the
other halves of BASELINE.json's metric measured the same way (C3 MIP, C3 with the nothing-skippable
table, C2, C4 and C5 at 9600 x 5400, C5 MIP), each cube generated, measured and freed in turn.

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
from dataclasses import replace

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_1012_2909_b200 import workloads as wl  # noqa: E402
from paper_1012_2909_b200.replicas import orbit_frame as _orbit_frame, reduce_run  # noqa: E402

METRIC = "ray samples/s (nominal lattice samples inside the cube; BASELINE.json metric)"
COUNTERS_JSON = os.path.join(ROOT, "profiles", "r2_counters.json")
ISSUE_SLOTS_PER_CLOCK = 148 * 4      # 148 SMs x 4 warp schedulers x 1 warp instruction per clock


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            return json.load(f), "measured (MEASURED_PEAKS.json)"
    return {"hbm_gbs": 6650.0}, "fallback (B200_PROFILING.md: 6.65 TB/s)"


def ncu_counters(workload, mode, tf, kernel):
    """Per-launch counters of the marcher from the committed ncu captures (profiles/r2_counters.json,
    written by `python -m paper_1012_2909_b200.ncu_counters`): nothing is typed into this file."""
    if not os.path.exists(COUNTERS_JSON):
        return None, "no capture: profiles/r2_counters.json is absent"
    with open(COUNTERS_JSON) as f:
        caps = json.load(f).get("captures", [])
    hits = [c for c in caps if c["workload"] == workload and c["mode"] == mode and c.get("tf") == tf and c["kernel"] in kernel]
    if not hits:
        return None, f"no capture of {kernel} for {workload} {mode} tf-{tf} in profiles/r2_counters.json"
    c = hits[-1]
    n = max(1, len(c["dram_bytes"]))
    return {"traffic": sum(c["dram_bytes"]) / n, "warp_instructions": sum(c["warp_instructions"]) / n, "frames": list(c.get("frames", [])),
            "launches": n, "source": f"{c['source']} (orbit frames {c.get('frames')}, {n} launches, commit {c.get('commit')})"}, None


def captured_frames(workload, mode, tf):
    """Orbit frames of the committed ncu captures of a workload (any kernel): the marcher is timed on them too, so that
    counters per launch and seconds per launch describe the same launches."""
    if not os.path.exists(COUNTERS_JSON):
        return []
    with open(COUNTERS_JSON) as f:
        caps = json.load(f).get("captures", [])
    return sorted({int(fr) for c in caps if c["workload"] == workload and c["mode"] == mode and c.get("tf") == tf for fr in c.get("frames", [])})


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


def kernel_name(plan, mode):
    """The marcher vr_render_bricks launches under a plan (vr_get_plan)."""
    v, skip, dense = plan["variant"], plan["skip_level"], plan["dense"]
    m = "EA" if mode == "ea" else "MIP"
    if v == 5:
        return "mip_tiles_kernel (object order: tiles of 32x32x16 cells staged in shared memory by bulk asynchronous copies)"
    if v == 3:
        if mode == "ea" and skip >= 3:
            return "render_occ_kernel (lockstep: occupancy test, compaction, gather, fold)"
        return f"render_ls_kernel<{m}> (lockstep{', dense fold' if dense and mode == 'ea' else ''})"
    if v == 4 and mode == "ea" and skip >= 3:
        return "render_occ_kernel<BEAM> (dense rays: beam test against the occupancy words, occupancy test in step, compaction, gather, fold)"
    if v == 1:
        return f"render_bricks_kernel<{m}> (ray per thread, CTA per (brick, tile))"
    return f"render_tiles_kernel<{m}> (ray per thread, skip level {skip})"


class Job:
    """One rank's resident cube + context.  configure() picks mode / table / frame without regenerating."""

    def __init__(self, w, device, mode="ea", shard=None, dist=None, tf=None, voxel="f32"):
        import torch
        from paper_1012_2909_b200 import vr
        self.torch, self.vr, self.w, self.voxel = torch, vr, w, voxel
        torch.cuda.set_device(device)
        self.ctx = vr.Context(device)
        vt = vr.VOXEL_F16 if voxel == "f16" else vr.VOXEL_F32
        self.ctx.set_option(vr.OPT_VOXEL_TYPE, vt)
        self.shard, self.dist = None, dist
        if shard is not None:                     # (rank, world): this rank holds one z-slab of the bricks
            from paper_1012_2909_b200 import sortlast
            self.sortlast = sortlast
            self.shard = sortlast.Shard(self.ctx, w.dims, w.brick, shard[0], shard[1])
            self.shard.bind()
            cb, mb = vr.cube_layout_typed(w.dims, w.brick, vt, self.shard.first, self.shard.end)
        else:
            cb, mb = vr.cube_layout_typed(w.dims, w.brick, vt)
        self.d_cube = torch.empty(max(cb // 4, 1), dtype=torch.float32, device="cuda")
        self.d_meta = torch.empty(max(mb, 1), dtype=torch.uint8, device="cuda")
        t0 = time.perf_counter()
        self.ctx.generate_cube(w.seed, w.dims, w.brick, self.d_cube, self.d_meta, sources=wl.make_sources(w),
                               zero_boxes=wl.make_zero_boxes(w), continuum=w.continuum)
        torch.cuda.synchronize()
        self.gen_seconds = time.perf_counter() - t0
        self.arena = None
        self.bitmap = None
        self.bg = (0.0, 0.0, 0.0, 0.0)
        self.slab_only = False
        self.staged = False
        self.peerfold = None
        self.streams = self.arenas = None
        self.configure(mode, tf or w.tf, w.frame, w.panels)

    def configure(self, mode, tf_name, frame, panels):
        torch, vr = self.torch, self.vr
        self.mode_name, self.tf_name = mode, tf_name
        self.mode = vr.MODE_EA if mode == "ea" else vr.MODE_MIP
        self.px_bytes = 16 if mode == "ea" else 4
        self.tf = wl.TFS[tf_name]()
        self.ctx.set_transfer_function(*self.tf)
        self.W, self.H = frame
        self.cols, self.rows = panels
        self.pw, self.ph = self.W // self.cols, self.H // self.rows
        ch = 4 if mode == "ea" else 1
        self.frame = None
        self.h_frame = None
        self.frame = torch.zeros((self.H, self.W, ch), dtype=torch.float32, device="cuda")
        self.h_frame = torch.empty((self.H, self.W, ch), dtype=torch.float32).pin_memory()
        self.reset_events()

    def reset_events(self):
        self.step_events, self.march_events, self.fold_events = [], [], []
        self.b_brick = self.partial_bytes = 0

    def close(self):
        self.ctx.close()
        self.d_cube = self.d_meta = self.arena = self.arenas = self.bitmap = self.frame = self.h_frame = None
        self.torch.cuda.empty_cache()

    def _arena(self, nbytes):
        if self.arena is None or self.arena.numel() < nbytes:
            self.arena = None
            self.arena = self.torch.empty(int(nbytes * 1.25) + 256, dtype=self.torch.uint8, device="cuda")
        return self.arena

    def brick_voxels(self):
        n = 1
        for b, d in zip(self.w.brick, self.w.dims):
            n *= min(b, d)
        return n

    def panel_views(self, frame_index):
        M = wl.config_camera(self.w, frame_index, frame=(self.W, self.H))
        for r in range(self.rows):
            for c in range(self.cols):
                yield c, r, (M if (self.cols, self.rows) == (1, 1) else wl.panel_matrix(M, self.cols, self.rows, c, r))

    def step(self, frame_index, timed_events=False, set_tf=False, one_call=False):
        """S1 + S2-S5 (+ S6) for one frame, sort-last path."""
        w, vr, ctx, torch = self.w, self.vr, self.ctx, self.torch
        if set_tf:
            ctx.set_transfer_function(*self.tf)
        if self.shard is not None:
            # sharded sort-last (paper_1012_2909_b200/sortlast.py): own bricks -> one partial frame; then ONE kernel reads
            # this rank's strip of every rank's partial frame through peer pointers, folds the versions in the slabs'
            # visibility order and stores the rows into every rank's final frame (--staged: all_to_all + fold + all_gather)
            sh, sl = self.shard, self.sortlast
            ctx.set_view(wl.config_camera(w, frame_index, frame=(self.W, self.H)), self.W, self.H, w.step)
            if self.peerfold is None or self.peerfold.mode != self.mode:
                self.peerfold = sl.PeerFold(sh, torch, self.mode, self.W, self.H, dist=self.dist)
            pf = self.peerfold
            ev = [torch.cuda.Event(enable_timing=True) for _ in range(4)] if timed_events else None
            if ev:
                ev[0].record()
            part = pf.render(w.tau)
            if ev:
                ev[1].record()
                self.march_events.append((ev[0], ev[1], frame_index))
                self.b_brick += 4 * self.brick_voxels() * (sh.end - sh.first)
                self.partial_bytes += self.H * self.W * self.px_bytes
            if self.slab_only:
                self.frame = part
            elif self.staged:
                versions = sl.exchange_strips(self.dist, part, sh.world)
                strip = sh.fold_strip(torch, self.mode, versions, self.W, self.H, self.bg)
                self.frame = sl.gather_strips(self.dist, strip, sh.world, self.H)
            else:
                pf.barrier()
                if ev:
                    ev[2].record()
                pf.fold(self.bg)
                if ev:
                    ev[3].record()
                    self.fold_events.append((ev[2], ev[3]))
                pf.barrier()
                self.frame = pf.final
            if timed_events:
                e = torch.cuda.Event(enable_timing=True)
                e.record()
                self.step_events.append(e)
            return
        if one_call:
            # the frame through vr_render_sortlast: sort, layout, march and fold of a panel in ONE call.  The panels of a
            # tiled frame write disjoint viewports: they go round-robin over 3 streams (each with its own arena), so the tail
            # of one panel's launch overlaps the next panel's; the first panel runs on the caller's stream and the others
            # start after it (it enqueues whatever a new table needs)
            main = torch.cuda.current_stream()
            multi = self.cols * self.rows > 1
            if multi and self.streams is None:
                self.streams = [torch.cuda.Stream() for _ in range(3)]
                self.arenas = [None, None, None]
            first = None
            for i, (c, r, Mp) in enumerate(self.panel_views(frame_index)):
                ctx.set_view(Mp, self.pw, self.ph, w.step)
                ctx.set_viewport(c * self.pw, r * self.ph, self.W)
                if not multi or i == 0:
                    st, slot = main, None
                else:
                    slot = i % 3
                    st = self.streams[slot]
                    st.wait_event(first)
                arena = self.arena if slot is None else self.arenas[slot]
                ok, need = ctx.render_sortlast(self.mode, arena, self.frame, self.bg, w.tau, stream=st.cuda_stream)
                if not ok:
                    arena = torch.empty(int(need * 1.25) + 256, dtype=torch.uint8, device="cuda")
                    if slot is None:
                        self.arena = arena
                    else:
                        self.arenas[slot] = arena
                    ok, need = ctx.render_sortlast(self.mode, arena, self.frame, self.bg, w.tau, stream=st.cuda_stream)
                    assert ok
                if multi and i == 0:
                    first = torch.cuda.Event()
                    first.record(main)
            if multi:
                for st in self.streams:
                    main.wait_stream(st)
            if timed_events:
                e = torch.cuda.Event(enable_timing=True)
                e.record()
                self.step_events.append(e)
            return
        for c, r, Mp in self.panel_views(frame_index):
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
                self.march_events.append((e0, e1, frame_index))
                # B_brick of this launch: the active in-frustum bricks read once;
                # nbytes: the partial images written once (16 or 4 B per pixel)
                self.b_brick += 4 * self.brick_voxels() * n
                self.partial_bytes += nbytes
            ctx.composite_bricks(self.mode, parts, n, self.frame, self.bg)
        if timed_events:
            e = torch.cuda.Event(enable_timing=True)
            e.record()
            self.step_events.append(e)

    def touch(self, frame_index):
        """B_touch of every vr_render_bricks launch of one frame: distinct 32-byte sectors and
        128-byte lines under the footprints of the samples the frame interpolates.  Untimed."""
        vr, ctx, torch, w = self.vr, self.ctx, self.torch, self.w
        if self.shard is not None:
            return None
        out = {"launches": 0, "sectors": 0, "lines": 0, "taken_samples": 0}
        for c, r, Mp in self.panel_views(frame_index):
            ctx.set_view(Mp, self.pw, self.ph, w.step)
            ctx.set_viewport(c * self.pw, r * self.ph, self.W)
            ids = ctx.sort_bricks(self.mode)
            parts, n, nbytes = ctx.partial_layout(self.mode, ids)
            vr.Context.bind_partials(parts, n, self._arena(nbytes))
            if self.bitmap is None:
                self.bitmap = torch.empty(ctx.touch_layout(), dtype=torch.uint8, device="cuda")
            ctx.measure_touch(self.mode, parts, n, self.bitmap, w.tau)
            t = ctx.touch_count(self.bitmap)
            out["launches"] += 1
            for k in ("sectors", "lines", "taken_samples"):
                out[k] += t[k]
        return out


def fetch_bricks(job, M, W, H, pix, cache):
    """Cube bytes of the bricks the rays of `pix` meet, fetched back from the device (untimed)."""
    from oracle import ovr
    w, torch = job.w, job.torch
    brick = tuple(min(b, n) for b, n in zip(w.brick, w.dims))
    touched = ovr.bricks_touched(M, W, H, w.step, w.dims, brick, pix)
    g = [-(-n // b) for n, b in zip(w.dims, brick)]
    for b in touched:
        if int(b) in cache:
            continue
        bi = (b % g[0], (b // g[0]) % g[1], b // (g[0] * g[1]))
        ext = [min(bb, n - i * bb) for i, bb, n in zip(bi, brick, w.dims)]
        t = torch.empty(ext[0] * ext[1] * ext[2], dtype=torch.float32, device="cuda")
        job.ctx.download_brick(int(b), t)
        cache[int(b)] = t.cpu().numpy()
    torch.cuda.synchronize()
    return ovr.Volume(w.dims, brick, {int(b): cache[int(b)] for b in touched}), brick, len(touched)


def oracle_sample(job, frame_index, tile, precision_name="F64", threads=1, cache=None):
    """Time the oracle, as it stands, on a tile x tile pixel block at the frame centre of the same frame
    (sort-last semantics, same partition, same tau).  threads > 1: the same code over disjoint interleaved
    pixel subsets on that many host threads (the ctypes call releases the GIL).  Returns (seconds, counters, bricks)."""
    from oracle import ovr
    w = job.w
    M = wl.config_camera(w, frame_index, frame=(job.W, job.H))
    cx, cy = job.W // 2, job.H // 2
    xs = np.arange(max(0, cx - tile // 2), min(job.W, cx - tile // 2 + tile))
    ys = np.arange(max(0, cy - tile // 2), min(job.H, cy - tile // 2 + tile))
    pix = np.stack(np.meshgrid(xs, ys), axis=-1).reshape(-1, 2).astype(np.int32)
    vol, brick, nb = fetch_bricks(job, M, job.W, job.H, pix, {} if cache is None else cache)
    omode = ovr.EA if job.mode == job.vr.MODE_EA else ovr.MIP

    def run(sub):
        _, _, cnt = ovr.render(vol, M, job.W, job.H, w.step, omode, getattr(ovr, precision_name), tf=job.tf,
                               split=ovr.SPLIT_SORTLAST, partition=brick, tau=w.tau, bg=job.bg, pixels=sub)
        return cnt

    t0 = time.perf_counter()
    if threads <= 1:
        cnts = [run(pix)]
    else:
        from concurrent.futures import ThreadPoolExecutor
        with ThreadPoolExecutor(max_workers=threads) as pool:
            cnts = list(pool.map(run, [np.ascontiguousarray(pix[i::threads]) for i in range(threads)]))
    sec = time.perf_counter() - t0
    cnt = {k: sum(c[k] for c in cnts) for k in cnts[0]}
    return sec, cnt, nb


def cpu_baseline(job, frame_index, seconds):
    """The oracle as it stands on one host core, and the same code over disjoint pixels on all host cores
    (BASELINE.md section 3), each on a pixel block sized for about `seconds` of wall time."""
    cores = len(os.sched_getaffinity(0)) if hasattr(os, "sched_getaffinity") else (os.cpu_count() or 1)
    cache = {}
    out = {}
    for label, threads in (("one", 1), ("all", cores)):
        tile = 8
        sec, c, nb = oracle_sample(job, frame_index, tile, threads=threads, cache=cache)
        if c["nominal"] > 0 and sec > 0:
            tile2 = int(min(384, max(8, tile * math.sqrt(seconds / max(sec, 1e-3)))))
            if tile2 > tile:
                sec, c, nb = oracle_sample(job, frame_index, tile2, threads=threads, cache=cache)
                tile = tile2
        out[label] = {"value": c["nominal"] / sec if sec > 0 else 0.0, "unit": "samples/s", "cores": threads, "kind": "oracle",
                      "sample": f"fp64 oracle, sort-last, the {tile}x{tile}-pixel block at the centre of orbit frame {frame_index} "
                                f"({c['nominal']} nominal samples, {nb} bricks fetched back from the device, {sec:.2f} s)"}
    res = out["one"]
    res["all_cores"] = out["all"]
    res["nproc"] = cores
    return res


def measure(job, steps, warmup, frank, fworld, dist, local_rank, e2e=True):
    """W untimed + K timed frames (device time, CUDA events), then the same K frames end to end with host buffers."""
    torch, w = job.torch, job.w

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    one = job.shard is None            # frames through vr_render_sortlast (the sharded path has its own calls)
    for i in range(warmup):
        job.step(orbit_frame(w, i, steps, frank, fworld), one_call=one)
    job.ctx.reset_counters()
    job.reset_events()
    sampler = ClockSampler(local_rank)
    barrier()
    sampler.start()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev0.record()
    for i in range(steps):
        torch.cuda.nvtx.range_push(f"timed_frame_{i}")       # ncu --nvtx --nvtx-include "timed_frame_0/": the launches of one whole frame
        job.step(orbit_frame(w, i, steps, frank, fworld), timed_events=True, one_call=one)
        torch.cuda.nvtx.range_pop()
    ev1.record()
    barrier()
    clocks = sampler.result()
    ms_total = ev0.elapsed_time(ev1)
    marks = [ev0] + job.step_events
    frame_ms = sorted(a.elapsed_time(b) for a, b in zip(marks, marks[1:]))
    cnt = job.ctx.get_counters()
    if one:
        # the marcher timed alone (roofline.launch_ms): the same frames through the separate calls, one launch after
        # the other on one stream, CUDA events around every vr_render_bricks
        job.reset_events()
        for i in range(min(steps, 6)):
            job.step(orbit_frame(w, i, steps, frank, fworld), timed_events=True)
        torch.cuda.synchronize()
        job.ctx.reset_counters()
    march_ms = sum(a.elapsed_time(b) for a, b, _ in job.march_events)
    n_march = len(job.march_events)
    by_frame = {}
    if one:
        # ... and on the orbit frames of the committed ncu captures (roofline.traffic / roofline.issue divide counters of
        # those launches by seconds of the same launches); kept apart from the means above
        keep = (job.march_events, job.b_brick, job.partial_bytes)
        job.reset_events()
        for f in captured_frames(w.name, job.mode_name, job.tf_name):
            job.step(f, timed_events=True)
        torch.cuda.synchronize()
        for a, b, f in job.march_events:
            by_frame.setdefault(f, []).append(a.elapsed_time(b))
        job.march_events, job.b_brick, job.partial_bytes = keep
        job.ctx.reset_counters()
    ms_total, (nominal, taken, launches) = reduce_run(
        dist, "cuda", ms_total, [cnt["nominal_samples"], cnt["taken_samples"], cnt["kernel_launches"]])
    res = {"ms_total": ms_total, "frame_ms": frame_ms, "nominal": nominal, "taken": taken, "launches": launches,
           "launches_per_step": n_march / max(1, min(steps, 6) if one else steps),
           "march_ms": march_ms, "n_march": n_march, "b_brick": job.b_brick, "partial_bytes": job.partial_bytes,
           "march_by_frame": by_frame, "clocks": clocks, "steps": steps, "fworld": fworld}
    if not e2e:
        return res
    # ---- e2e: the same step through the public API with HOST buffers in the timed region: the
    # view matrix and the transfer-function table go host -> device every step (as kernel
    # parameters / table upload), the finished frame comes back device -> pinned host memory.
    # Two frame buffers: frame i's device -> host copy runs on a copy stream while frame i + 1 is rendered;
    # the host takes delivery of frame i - 1 (waits for its copy) before it issues frame i + 1.
    job.ctx.reset_counters()
    barrier()
    frames = [job.frame, torch.zeros_like(job.frame)]
    h_frames = [job.h_frame, torch.empty_like(job.h_frame).pin_memory()]
    copy_stream = torch.cuda.Stream()
    copied = [None, None]
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for i in range(steps):
        b = i % 2
        if copied[b] is not None:
            torch.cuda.current_stream().wait_event(copied[b])      # the buffer's previous frame has left the device
        job.frame = frames[b]
        job.step(orbit_frame(w, i, steps, frank, fworld), set_tf=True, one_call=True)
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
    copied[(steps - 1) % 2].synchronize()
    torch.cuda.synchronize()
    e2e_s = time.perf_counter() - t0
    job.frame = frames[0]
    cnt2 = job.ctx.get_counters()
    e2e_s, (e2e_nominal,) = reduce_run(dist, "cuda", e2e_s, [cnt2["nominal_samples"]])
    res["e2e_s"], res["e2e_nominal"] = e2e_s, e2e_nominal
    return res


def roofline(job, m, touch_frames, peak, peak_src):
    """algorithmic bytes per launch = min(B_brick, B_touch) + partial images written + brick meta,
    over the launch's CUDA-event duration.  B_touch is measured by vr_measure_touch on `touch_frames`."""
    n = max(m["n_march"], 1)
    launch_s = m["march_ms"] / n * 1e-3
    plan = job.ctx.get_plan(job.mode)
    kernel = kernel_name(plan, job.mode_name)
    b_brick = m["b_brick"] / n
    writes = m["partial_bytes"] / n + 8 * job.w.brick_grid[0] * job.w.brick_grid[1] * job.w.brick_grid[2]
    touch = None
    if touch_frames:
        acc = {"launches": 0, "sectors": 0, "lines": 0, "taken_samples": 0}
        for f in touch_frames:
            t = job.touch(f)
            if t is None:
                acc = None
                break
            for k in acc:
                acc[k] += t[k]
        if acc and acc["launches"]:
            touch = {"frames": list(touch_frames), "sector_bytes_per_launch": 32.0 * acc["sectors"] / acc["launches"],
                     "line_bytes_per_launch": 128.0 * acc["lines"] / acc["launches"],
                     "taken_samples_per_launch": acc["taken_samples"] / acc["launches"]}
    b_touch = touch["sector_bytes_per_launch"] if touch else None
    alg = (min(b_brick, b_touch) if b_touch is not None else b_brick) + writes
    achieved = alg / launch_s / 1e9 if launch_s > 0 else 0.0
    out = {"bound": "hbm", "kernel": kernel, "achieved": achieved, "peak": peak, "unit": "GB/s",
           "frac": achieved / peak if peak else None, "peak_source": peak_src,
           "algorithmic_bytes_per_launch": alg, "b_brick": b_brick, "b_touch": touch, "bytes_written": writes,
           "launch_ms": m["march_ms"] / n, "launches_per_step": m["launches_per_step"],
           "share_of_step": min(1.0, m["march_ms"] / n * m["launches_per_step"] / (m["ms_total"] / m["steps"])) if m["ms_total"] else None,
           "plan": plan,
           "effective_vs_brick": (b_brick + writes) / launch_s / 1e9 / peak if launch_s > 0 and peak else None,
           "note": "algorithmic bytes = min(B_brick, B_touch) + partial images + brick meta (SURVEY.md 8(d)); B_brick = 4 B x "
                   "voxels of the active in-frustum bricks at the configured size; B_touch = 32 B x distinct sectors under the "
                   "footprints of the samples the launch interpolates (vr_measure_touch on the frames listed); frac_lines "
                   "counts whole 128-byte lines instead (the unit this HBM is read in, DESIGN.md section 4); "
                   "effective_vs_brick is the B_brick ratio (can exceed 1: skipping below the brick level)"}
    if touch:
        lines = min(b_brick, touch["line_bytes_per_launch"]) + writes
        out["frac_lines"] = lines / launch_s / 1e9 / peak if launch_s > 0 and peak else None
    cap, why = ncu_counters(job.w.name, job.mode_name, job.tf_name, kernel)
    clocks = m["clocks"]
    if cap:
        # seconds per launch of the very launches that were captured: the same orbit frames, timed alone in this run (a tiled
        # frame: the first `launches` panels of the frame if fewer than all were captured - named in the capture's title)
        # (a panel that no brick meets launches nothing: the captured launches of a frame are fewer than its panels, so the
        # frames' summed marcher time is divided by the number of CAPTURED launches, which are whole frames)
        by = m.get("march_by_frame", {})
        have = all(f in by for f in cap["frames"]) and cap["frames"]
        cap_s = sum(t for f in cap["frames"] for t in by[f]) / cap["launches"] * 1e-3 if have else None
        out["traffic"] = cap["traffic"]
        out["traffic_source"] = cap["source"]
        out["captured_launch_ms"] = cap_s * 1e3 if cap_s else None
        if cap_s:
            out["dram_gbs_from_traffic"] = cap["traffic"] / cap_s / 1e9
            out["traffic_frac"] = out["dram_gbs_from_traffic"] / peak if peak else None      # what ncu saw the launch move, over the HBM peak
            if clocks.get("sm_mhz"):
                ipeak = ISSUE_SLOTS_PER_CLOCK * clocks["sm_mhz"] * 1e6 / 1e9
                out["issue"] = {"bound": "alu", "achieved": cap["warp_instructions"] / cap_s / 1e9, "peak": ipeak,
                                "unit": "G warp-instructions/s", "frac": cap["warp_instructions"] / cap_s / 1e9 / ipeak,
                                "note": "warp instructions per launch from the committed ncu capture / seconds per launch of the same orbit "
                                        "frames timed alone in this run; peak = 148 SMs x 4 schedulers x the SM clock sampled during the run"}
        else:
            out["traffic_note"] = "the captured orbit frames were not timed in this run (sharded / slab runs): no rate derived from the capture"
    else:
        out["traffic"] = None
        out["traffic_note"] = why
    return out


def entry(job, m, args, peak, peak_src, touch_frames):
    """The JSON fields of one measured workload."""
    steps, fworld, ms_total = m["steps"], m["fworld"], m["ms_total"]
    frame_ms = m["frame_ms"]
    w = job.w
    out = {
        "value": m["nominal"] / (ms_total * 1e-3), "unit": "samples/s", "steps": steps,
        "ms_per_step": ms_total / steps, "frames_per_s": steps * fworld / (ms_total * 1e-3),
        "frame_ms": {"median": frame_ms[len(frame_ms) // 2], "p95": frame_ms[min(len(frame_ms) - 1, int(0.95 * len(frame_ms)))],
                     "min": frame_ms[0], "max": frame_ms[-1], "note": "rank 0, device time between consecutive frames of the orbit"},
        "nominal_samples_per_step": m["nominal"] / (steps * fworld),
        "taken_samples_per_s": m["taken"] / (ms_total * 1e-3),
        "taken_fraction": m["taken"] / max(m["nominal"], 1),
        "gpu_launches": m["launches"],
        "clocks": m["clocks"],
        "roofline": roofline(job, m, touch_frames, peak, peak_src),
    }
    if "e2e_s" in m:
        out["e2e"] = {"value": m["e2e_nominal"] / m["e2e_s"], "unit": "samples/s", "ms_per_step": m["e2e_s"] * 1e3 / steps,
                      "h2d_bytes_per_step": (64 + 4096 + 8) * job.cols * job.rows,
                      "d2h_bytes_per_step": job.H * job.W * job.px_bytes}
    return out


def describe(job, mode, world, args):
    w = job.w
    return {"workload": f"{w.name}: {w.dims[0]}x{w.dims[1]}x{w.dims[2]} cube stored as {'float16' if job.voxel == 'f16' else 'float32'}, {w.brick[0]}^3 bricks, "
                        f"{job.W}x{job.H} frame ({job.cols}x{job.rows} panels), step {w.step}, "
                        f"{'EA tf-' + job.tf_name + ' tau=' + str(w.tau) if mode == 'ea' else 'MIP'}, sort-last path, orbit frames spread over 360 deg",
            "cube_gib": round(w.n_voxels * (2 if job.voxel == "f16" else 4) / 2 ** 30, 3), "n_sources": w.n_sources,
            "l2_policy": "inputs larger than L2 (cube >> 126 MB); no explicit flush",
            "e2e_policy": "through vr_set_view + vr_render_sortlast (one call per panel); matrix + table host->device and frame device->pinned host every step; two frame buffers, frame "
                          "i's copy overlaps frame i+1's render, the host waits for frame i-1 before issuing frame i+1",
            "replicas": 1 if args.sharded else world, "shards": world if args.sharded else 1, "slab": args.slab,
            "generate_seconds": round(job.gen_seconds, 3)}


def tf_edit(job, frame_index):
    """Milliseconds from a transfer-function edit that changes the SET of transparent entries (the opacity
    threshold dragged from entry 32 to 40 and back; "colour map", line 13 "interactive") to the
    finished next frame: vr_set_transfer_function + one step, stream synchronised (re-classification included)."""
    torch = job.torch
    keep = job.tf
    times = []
    for k in range(4):
        job.tf = wl.tf_src(40 if k % 2 == 0 else 32)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        job.step(frame_index, set_tf=True, one_call=True)
        torch.cuda.synchronize()
        times.append((time.perf_counter() - t0) * 1e3)
    job.tf = keep
    job.step(frame_index, set_tf=True)
    torch.cuda.synchronize()
    times.sort()
    return {"ms": times[len(times) // 2], "all_ms": times, "what": "threshold entry 32 <-> 40, then one frame, synchronised"}


SUITE = [  # (workload, mode, table, frame, panels, steps, voxels): the rest of BASELINE.json's metric, each measured like the headline
    ("C3", "mip", None, None, None, 12, "f32"),
    ("C3", "ea", "fog", None, None, 12, "f32"),
    ("C2", "ea", None, None, None, 24, "f32"),
    # (tiled frames: the end-to-end loop ends with one frame copy of 829 MB that overlaps nothing, ~19 ms spread over the
    # timed frames: 16 / 10 of them, so that the figure is the steady state's within ~1 ms)
    ("C4", "ea", None, None, None, 16, "f32"),
    ("C5", "ea", None, None, None, 10, "f32"),
    ("C5", "mip", None, (1920, 1080), (1, 1), 12, "f32"),
    # the paper's HIPASS shape, and a 256 GiB-class cube resident as float16
    ("HIPASS", "ea", None, None, None, 8, "f32"),
    ("W256", "ea", None, None, None, 8, "f16"),
    ("W256", "mip", None, None, None, 8, "f16"),
]


def run_suite(args, head_job, peak, peak_src, local_rank):
    import torch
    out = []
    job = head_job
    for name, mode, tf, frame, panels, steps, voxel in SUITE:
        w = wl.CONFIGS[name]
        try:
            if job is None or job.w.name != name or job.voxel != voxel:
                if job is not None:
                    job.close()
                    job = None
                free, _ = torch.cuda.mem_get_info()
                need = w.n_voxels * (2 if voxel == "f16" else 4) * (1.16 if voxel == "f16" else 1.10) + 3e9
                if free < need:
                    out.append({"config": {"workload": name, "mode": mode}, "skipped": f"needs {need / 1e9:.0f} GB of free HBM, {free / 1e9:.0f} free"})
                    continue
                job = Job(w, local_rank, mode, tf=tf, voxel=voxel)
            job.configure(mode, tf or w.tf, frame or w.frame, panels or w.panels)
            m = measure(job, steps, 3, 0, 1, None, local_rank)
            e = entry(job, m, args, peak, peak_src, [orbit_frame(w, 0, steps, 0, 1)] if not args.no_touch else [])
            e["config"] = describe(job, mode, 1, args)
            if name == "C2" and not args.no_cpu:
                e["cpu_baseline"] = cpu_baseline(job, orbit_frame(w, 0, steps, 0, 1), args.cpu_seconds / 2)
            out.append(e)
        except Exception as exc:                      # one failing entry must not lose the headline
            out.append({"config": {"workload": name, "mode": mode}, "error": f"{type(exc).__name__}: {exc}"})
            try:
                if job is not None:
                    job.close()
            except Exception:
                pass
            job = None
    if job is not None:
        job.close()
    try:                                              # the HIPASS-shaped cube streamed from pinned host memory
        out.append(run_streamed(wl.CONFIGS["HIPASS"], "ea", 2, 6, 2, local_rank))
    except Exception as exc:
        out.append({"config": {"workload": "HIPASS streamed"}, "error": f"{type(exc).__name__}: {exc}"})
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=24)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default=None, choices=sorted(wl.CONFIGS))
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--mode", default="ea", choices=["ea", "mip"], help="emission-absorption (default) or MIP")
    ap.add_argument("--tf", default=None, choices=sorted(wl.TFS), help="transfer function (default: the workload's)")
    ap.add_argument("--voxel", default="f32", choices=["f32", "f16"], help="stored voxel type (VR_OPT_VOXEL_TYPE)")
    ap.add_argument("--sharded", action="store_true",
                    help="N ranks share ONE cube: bricks sharded in z-slabs, sort-last exchange over NCCL (NEXT-1, "
                         "strong scaling); default: N independent replicas")
    ap.add_argument("--staged", action="store_true", help="--sharded with the staged exchange (all_to_all_single + fold + all_gather) "
                                                          "instead of the fused peer-memory kernel: the A/B baseline")
    ap.add_argument("--slab", default=None, metavar="R/W",
                    help="render only slab R of a W-way split of the bricks (what rank R of --sharded would render; no "
                         "exchange): the per-rank cost of NEXT-1 measured on one GPU")
    ap.add_argument("--next-rows", action="store_true",
                    help="time the catalogue overlay and the output pyramid (SURVEY.md 8(f) 2 and 3) instead of the marcher")
    ap.add_argument("--frame", default=None, help="WxH: render one frame of this size instead of the workload's "
                                                   "(BASELINE.json configs[4]: C5's 1920x1080 MIP)")
    ap.add_argument("--cpu-seconds", type=float, default=12.0, help="target wall time of each oracle sample")
    ap.add_argument("--suite", dest="suite", action="store_true", default=None,
                    help="append the `configs` list (default: on for the default workload on one GPU)")
    ap.add_argument("--no-suite", dest="suite", action="store_false")
    ap.add_argument("--no-cpu", action="store_true", help="skip the oracle timing (profiling runs)")
    ap.add_argument("--no-touch", action="store_true", help="skip the B_touch measurement (profiling runs)")
    ap.add_argument("--streamed", type=int, default=0, metavar="SLOTS",
                    help="out-of-core run: the cube in pinned host memory, streamed through SLOTS device slots of one slab each "
                         "(SURVEY.md 8(f)-4; paper_1012_2909_b200/outofcore.py)")
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

    default_run = (args.workload is None and args.mode == "ea" and args.tf is None and not args.frame and not args.sharded
                   and not args.slab and world == 1 and args.voxel == "f32")
    if args.suite is None:
        args.suite = default_run and args.impl == "b200"
    w = wl.CONFIGS[args.workload or "C3"]
    if args.frame:
        w = replace(w, frame=tuple(int(v) for v in args.frame.lower().split("x")), panels=(1, 1))
    if args.next_rows:
        return run_next_rows(args)
    if args.streamed:
        print(json.dumps(run_streamed(w, args.mode, args.streamed, args.steps, args.warmup, local_rank, args.tf, args.voxel)))
        return 0
    slab = None
    if args.slab:
        slab = tuple(int(v) for v in args.slab.split("/"))
        if world != 1 or args.sharded or not (0 <= slab[0] < slab[1]):
            raise SystemExit("--slab R/W runs on one GPU, without --sharded")
    if (args.sharded or slab) and w.panels != (1, 1):
        raise SystemExit("--sharded renders single-panel frames (use --frame WxH for the tiled workloads)")
    job = Job(w, local_rank, args.mode, shard=slab if slab else ((rank, world) if args.sharded else None), dist=dist, tf=args.tf,
              voxel=args.voxel)
    job.slab_only = slab is not None
    job.staged = args.staged
    frank, fworld = (0, 1) if args.sharded else (rank, world)          # sharded: every rank renders every frame
    config = describe(job, args.mode, world, args)

    if args.impl == "reference":
        return run_reference(args, job, config)

    m = measure(job, args.steps, args.warmup, frank, fworld, dist, local_rank)
    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return 0

    peaks, peak_src = measured_peaks()
    peak = float(peaks["hbm_gbs"])
    f0 = orbit_frame(w, 0, args.steps, 0, 1)
    touch_frames = [] if (args.no_touch or args.sharded or slab) else sorted({f0, orbit_frame(w, args.steps // 2, args.steps, 0, 1)})
    out = {"metric": METRIC}
    out.update(entry(job, m, args, peak, peak_src, touch_frames))
    out.update({"n_gpus": world, "warmup": args.warmup, "higher_is_better": True, "scaling": "strong" if args.sharded else "weak",
                "vs_baseline": None, "dtype": "f32", "data": "synthetic", "config": config})
    if args.sharded or slab:
        fold_ms = [a.elapsed_time(b) for a, b in job.fold_events]
        out["sharded"] = {"exchange": "staged (NCCL all_to_all_single + vr_composite_bricks + all_gather)" if args.staged else
                          "fused (vr_fold_peers: peer-pointer loads, over-operator, peer-pointer stores in one kernel)",
                          "rank0_render_ms": m["march_ms"] / max(m["n_march"], 1),
                          "rank0_fold_ms": sum(fold_ms) / len(fold_ms) if fold_ms else None,
                          "measured_on_ranks": world, "note": "N > 1 was not available to this build: unmeasured on hardware beyond what this line shows"}
    if world == 1 and not slab and not args.no_cpu:           # a slab holds only its own bricks: no oracle sample
        out["cpu_baseline"] = cpu_baseline(job, f0, args.cpu_seconds)
        out["vs_cpu_baseline"] = {"one_core": out["value"] / out["cpu_baseline"]["value"] if out["cpu_baseline"]["value"] else None,
                                  "all_cores": out["value"] / out["cpu_baseline"]["all_cores"]["value"] if out["cpu_baseline"]["all_cores"]["value"] else None,
                                  "note": "GPU device-timed rate over the oracle's: reported, not a headline (the oracle is a deliberately plain program)"}
    else:
        out["cpu_baseline"] = None
    if default_run and args.mode == "ea" and job.tf_name == "src":
        out["tf_edit"] = tf_edit(job, f0)
    if args.suite:
        out["configs"] = run_suite(args, job, peak, peak_src, local_rank)
    print(json.dumps(out))
    if dist is not None:
        dist.destroy_process_group()
    return 0


def run_streamed(w, mode_name, n_slots, steps, warmup, local_rank, tf_name=None, voxel="f32"):
    """SURVEY.md 8(f)-4 / PAPER.md line 19 (cubes "larger than a single machine memory limit"): the cube kept brick-major in
    pinned host memory, streamed per frame through `n_slots` device slots of one slab (whole z-layers of bricks) each
    (paper_1012_2909_b200/outofcore.py): host -> device copy of the next slab overlapping the render of the current one, one
    vr_fold_peers launch per frame.  Wall-clock per frame, synchronised (the copies are part of the frame)."""
    import torch
    from paper_1012_2909_b200 import outofcore, vr
    torch.cuda.set_device(local_rank)
    grid_z = -(-w.dims[2] // w.brick[2])
    t0 = time.perf_counter()
    cube = outofcore.StreamedCube(w.dims, w.brick, n_slabs=min(grid_z, 32), n_slots=n_slots, device=local_rank,
                                  voxel_type=vr.VOXEL_F16 if voxel == "f16" else vr.VOXEL_F32)
    cube.ingest_generated(w.seed, sources=wl.make_sources(w), zero_boxes=wl.make_zero_boxes(w), continuum=w.continuum)
    ingest_s = time.perf_counter() - t0
    mode = vr.MODE_EA if mode_name == "ea" else vr.MODE_MIP
    cube.set_transfer_function(*wl.TFS[tf_name or w.tf]())
    W, H = w.frame if w.panels == (1, 1) else (w.frame[0] // w.panels[0], w.frame[1] // w.panels[1])
    times = []
    for i in range(warmup + steps):
        M = wl.config_camera(w, orbit_frame(w, max(i - warmup, 0), steps, 0, 1), frame=(W, H))
        torch.cuda.synchronize()
        before = dict(cube.stats)
        t0 = time.perf_counter()
        cube.render(mode, M, W, H, w.step, tau=w.tau)
        torch.cuda.synchronize()
        if i >= warmup:
            times.append((time.perf_counter() - t0, cube.stats["h2d_bytes"] - before["h2d_bytes"], cube.stats["slabs_copied"] - before["slabs_copied"]))
    total_s = sum(t[0] for t in times)
    out = {"config": {"workload": f"{w.name} streamed: {w.dims[0]}x{w.dims[1]}x{w.dims[2]} {'float16' if voxel == 'f16' else 'float32'} cube in pinned host memory, "
                                  f"{cube.n_slabs} slabs of whole brick layers through {cube.n_slots} device slots, {W}x{H} frame, "
                                  f"{'EA tf-' + (tf_name or w.tf) if mode_name == 'ea' else 'MIP'}, step {w.step}",
                      "host_gib": round(cube.host_bytes() / 2 ** 30, 2),
                      "device_pool_gib": round(sum(s["d_cube"].numel() * 4 for s in cube.slots) / 2 ** 30, 2)},
           "ms_per_step": total_s * 1e3 / len(times), "frames_per_s": len(times) / total_s, "steps": len(times),
           "slabs_copied_per_frame": sum(t[2] for t in times) / len(times),
           "h2d_gb_per_frame": sum(t[1] for t in times) / len(times) / 1e9,
           "h2d_gbs": sum(t[1] for t in times) / total_s / 1e9,
           "ingest_seconds": round(ingest_s, 2),
           "note": "wall clock, synchronised per frame: the frame time is the host -> device traffic of the slabs that are not resident"}
    cube.close()
    return out


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
    cache = {}
    sec, c, nb = oracle_sample(job, 0, tile, cache=cache)
    if sec > 0:
        tile = int(min(128, max(4, tile * math.sqrt(budget / max(sec, 1e-3)))))
    for i in range(args.warmup):
        oracle_sample(job, orbit_frame(w, i, args.steps, 0, 1), tile, cache=cache)
    total_s, total_n = 0.0, 0
    for i in range(args.steps):
        sec, c, nb = oracle_sample(job, orbit_frame(w, i, args.steps, 0, 1), tile, cache=cache)
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
