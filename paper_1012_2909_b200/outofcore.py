"""Rendering a cube that does not fit in HBM (section 1: "capable of volume
rendering image cubes larger than a single machine memory limit", line 47: the WALLABY cube).

The paper spreads the sub-volumes over the memories of several GPUs and composites their images; one B200 can do
the same IN TIME instead of in space.  The cube lives brick-major in pinned host memory, cut into slabs of whole
z-layers of bricks (the slabs of paper_1012_2909_b200/sortlast.py); a small pool of device slots holds a few slabs at a time.
Per frame the slabs that meet the frustum are visited one after the other (in alternating direction from frame to frame,
so that the slabs the last frame left resident come first): the next slab is copied host -> device on
a copy stream while the current one is rendered into its own premultiplied partial frame (`vr_render_bricks` +
`vr_composite_bricks` on the resident window, `vr_set_brick_window`), and ONE `vr_fold_peers` launch folds the
slabs' partial frames in the slabs' visibility order (`vr_sort_groups`) and adds the background - the very fold of
the multi-GPU path, so a streamed frame equals the frame of the same slabs spread over GPUs bit for bit, and the
oracle's two-level composite (tests/test_gpu_outofcore.py).

A slab that is still resident from the previous frame is not copied again; a slab entering a slot is attached with
`vr_attach_cube`: its cube bytes and the leading, table-independent part of its metadata (`vr_meta_static_bytes`)
come from the host, the classification against the transfer function is recomputed on the device by the next render.

Marshalling and residency only (copies, windows, which slab goes where): every arithmetic step runs in libvr's kernels.
"""
from __future__ import annotations

import numpy as np

from . import sortlast, vr


class StreamedCube:
    """A cube in pinned host memory rendered through `n_slots` device slots of one slab each."""

    def __init__(self, dims, brick, n_slabs: int, n_slots: int = 2, device: int = 0, voxel_type: int = vr.VOXEL_F32,
                 options=None):
        import torch
        self.torch = torch
        self.dims, self.brick = tuple(int(v) for v in dims), tuple(int(v) for v in brick)
        self.grid = [-(-n // min(b, n)) for n, b in zip(self.dims, self.brick)]
        self.n_slabs = max(1, min(int(n_slabs), self.grid[2], 32))          # vr_fold_peers folds up to 32 partial frames
        self.group_first = sortlast.slab_groups(self.grid, self.n_slabs)
        self.n_slots = max(1, min(int(n_slots), self.n_slabs))
        self.voxel_type, self.device = int(voxel_type), int(device)
        torch.cuda.set_device(self.device)
        self.sizes = []                                                      # per slab: (cube bytes, meta bytes, static meta bytes)
        for g in range(self.n_slabs):
            first, end = self.group_first[g], self.group_first[g + 1]
            cb, mb = vr.cube_layout_typed(self.dims, self.brick, self.voxel_type, first, end)
            self.sizes.append((cb, mb, vr.meta_static_bytes(self.dims, self.brick, self.voxel_type, first, end)))
        cb_max, mb_max = max(s[0] for s in self.sizes), max(s[1] for s in self.sizes)
        self.slots = []
        for _ in range(self.n_slots):
            ctx = vr.Context(self.device)
            ctx.set_option(vr.OPT_VOXEL_TYPE, self.voxel_type)
            for opt, value in (options or {}).items():
                ctx.set_option(opt, value)
            self.slots.append({"ctx": ctx, "slab": -1, "attached": -1, "shard": None,
                               "d_cube": torch.empty(max(cb_max // 4, 64), dtype=torch.float32, device="cuda"),
                               "d_meta": torch.empty(max(mb_max, 256), dtype=torch.uint8, device="cuda"),
                               "copied": torch.cuda.Event(), "rendered": torch.cuda.Event()})
        self.geometry = vr.Context(self.device)                              # no brick resident: screen rectangles and slab order only
        self.geometry.set_option(vr.OPT_VOXEL_TYPE, self.voxel_type)
        self.geometry.set_brick_window(0, 0)
        self._dummy = torch.zeros(256, dtype=torch.uint8, device="cuda")
        self.geometry.attach_cube(self.dims, self.brick, self._dummy, self._dummy)
        self.copy_stream = torch.cuda.Stream()
        self.h_cube = [None] * self.n_slabs                                  # pinned host copies, brick-major
        self.h_meta = [None] * self.n_slabs
        self.tf = None
        self.partials = {}
        self.final = None
        self.stats = {"frames": 0, "slabs_rendered": 0, "slabs_copied": 0, "h2d_bytes": 0}

    # ------------------------------------------------------------------ ingest: device -> pinned host, slab by slab
    def _bind(self, slot, g):
        slot["ctx"].set_brick_window(self.group_first[g], self.group_first[g + 1])

    def _save(self, slot, g):
        torch = self.torch
        cb, _, sb = self.sizes[g]
        self.h_cube[g] = torch.empty(max(cb // 4, 1), dtype=torch.float32).pin_memory()
        self.h_meta[g] = torch.empty(max(sb, 1), dtype=torch.uint8).pin_memory()
        self.h_cube[g].copy_(slot["d_cube"][:self.h_cube[g].numel()])
        self.h_meta[g].copy_(slot["d_meta"][:self.h_meta[g].numel()])
        torch.cuda.synchronize()
        slot["slab"], slot["attached"] = g, g                                # what it holds now: generated and classified in place

    def ingest_generated(self, seed, sources=None, zero_boxes=None, continuum=0.0):
        """The synthetic cube (vr_generate_cube), one slab at a time through slot 0."""
        slot = self.slots[0]
        for g in range(self.n_slabs):
            self._bind(slot, g)
            slot["ctx"].generate_cube(seed, self.dims, self.brick, slot["d_cube"], slot["d_meta"], sources=sources,
                                      zero_boxes=zero_boxes, continuum=continuum)
            self._save(slot, g)

    def ingest_host(self, cube):
        """A linear host cube [nz, ny, nx] (numpy, may be a memory map), one slab at a time through slot 0."""
        slot = self.slots[0]
        for g in range(self.n_slabs):
            self._bind(slot, g)
            slot["ctx"].upload_cube(cube, self.dims, self.brick, slot["d_cube"], slot["d_meta"])
            self._save(slot, g)

    def host_bytes(self):
        return sum(t.numel() * t.element_size() for t in self.h_cube + self.h_meta if t is not None)

    # ------------------------------------------------------------------ per frame
    def set_transfer_function(self, rgba, vmin, vmax):
        self.tf = (rgba, vmin, vmax)
        for slot in self.slots:
            slot["ctx"].set_transfer_function(rgba, vmin, vmax)

    def _needed(self, mode, M, W, H, step):
        """Slabs with a brick in the frustum, in the slabs' visibility order (geometry only)."""
        geo = self.geometry
        geo.set_view(M, W, H, step)
        order = [int(g) for g in geo.sort_groups(self.group_first)]
        ids = np.arange(self.grid[0] * self.grid[1] * self.grid[2], dtype=np.int32)
        parts, n, _ = geo.partial_layout(mode, ids)
        seen = np.zeros(self.n_slabs, dtype=bool)
        firsts = np.asarray(self.group_first)
        for i in range(n):
            seen[np.searchsorted(firsts, parts[i].brick, side="right") - 1] = True
        return [g for g in order if seen[g]], order

    def _prefetch(self, g, keep):
        """Make slab g resident (copy stream), evicting a slot whose slab is not in `keep`."""
        for slot in self.slots:
            if slot["slab"] == g:
                return slot
        torch = self.torch
        victims = [s for s in self.slots if s["slab"] not in keep]
        slot = victims[0] if victims else None
        if slot is None:
            return None
        with torch.cuda.stream(self.copy_stream):
            self.copy_stream.wait_event(slot["rendered"])                    # the slot's last render has read it
            hc, hm = self.h_cube[g], self.h_meta[g]
            slot["d_cube"][:hc.numel()].copy_(hc, non_blocking=True)
            slot["d_meta"][:hm.numel()].copy_(hm, non_blocking=True)
            slot["copied"].record(self.copy_stream)
        slot["slab"] = g
        self.stats["slabs_copied"] += 1
        self.stats["h2d_bytes"] += hc.numel() * 4 + hm.numel()
        return slot

    def render(self, mode, M, W, H, step, bg=(0.0, 0.0, 0.0, 0.0), tau=0.99):
        """One frame [H, W, 4] (EA) or [H, W, 1] (MIP; bg[0] = the miss value)."""
        torch = self.torch
        assert self.tf is not None and all(t is not None for t in self.h_cube), "ingest a cube and set a transfer function first"
        ch = 4 if mode == vr.MODE_EA else 1
        if self.final is None or tuple(self.final.shape) != (H, W, ch):
            self.final = torch.zeros((H, W, ch), dtype=torch.float32, device="cuda")
            self.partials = {}
        main = torch.cuda.current_stream()
        needed, order = self._needed(mode, M, W, H, step)
        # The fold at the end takes the partial frames in visibility order whatever order they were rendered in, so the
        # slabs are VISITED in the direction that meets the resident ones first: front to back on one frame, back to
        # front on the next (visiting them the same way round every frame evicts each slab just before it is wanted again).
        resident = {s["slab"] for s in self.slots}
        back = needed[::-1]
        seq = needed if sum(g in resident for g in needed[:self.n_slots]) >= sum(g in resident for g in back[:self.n_slots]) else back
        for i, g in enumerate(seq):
            window = seq[i:i + self.n_slots]                                 # slabs that must not be evicted now
            slot = self._prefetch(g, window)
            for nxt in seq[i + 1:i + self.n_slots]:                          # copies of the next slabs overlap this render
                self._prefetch(nxt, window)
            main.wait_event(slot["copied"])
            ctx = slot["ctx"]
            if slot["attached"] != g:
                self._bind(slot, g)
                ctx.attach_cube(self.dims, self.brick, slot["d_cube"], slot["d_meta"])
                slot["attached"] = g
                slot["shard"] = None
            if slot["shard"] is None:
                slot["shard"] = sortlast.Shard(ctx, self.dims, self.brick, g, self.n_slabs, group_first=self.group_first)
            ctx.set_view(M, W, H, step)
            if g not in self.partials:
                self.partials[g] = torch.empty((H, W, ch), dtype=torch.float32, device="cuda")
            slot["shard"].render_partial(torch, mode, W, H, tau, out=self.partials[g])
            slot["rendered"].record(main)
            self.stats["slabs_rendered"] += 1
        # one fold of the slabs' partial frames, in the slabs' order, plus the background (vr_fold_peers on one "rank")
        frames = [self.partials[g] for g in order if g in needed]
        if not frames:                                                       # nothing in the frustum: an empty partial frame
            if "empty" not in self.partials:
                self.partials["empty"] = torch.full((H, W, ch), 0.0 if mode == vr.MODE_EA else float("-inf"),
                                                    dtype=torch.float32, device="cuda")
            frames = [self.partials["empty"]]
        fold_bg = bg if mode == vr.MODE_EA else (bg[0], 0.0, 0.0, 0.0)
        self.slots[0]["ctx"].fold_peers(mode, [f.data_ptr() for f in frames], list(range(len(frames))), W, H, W, 0, H,
                                        [self.final.data_ptr()], W, fold_bg)
        self.stats["frames"] += 1
        return self.final

    def close(self):
        for slot in self.slots:
            slot["ctx"].close()
        self.geometry.close()
        self.slots, self.h_cube, self.h_meta, self.partials, self.final = [], [], [], {}, None
        self.torch.cuda.empty_cache()
