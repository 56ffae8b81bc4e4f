"""Sort-last rendering with the bricks sharded over several GPUs.

PAPER.md line 13 (abstract) and line 19 (section 1): the framework renders sub-volumes on
"distributed GPUs" and composites their images.  Here rank r of `world` holds one slab of whole
z-layers of bricks (`vr_set_brick_window`), renders the partial images of its resident bricks and
folds them into ONE premultiplied partial frame (`vr_render_bricks` + `vr_composite_bricks`); the
frame is then cut into `world` strips of rows, every rank receives all versions of its strip
(direct-send all-to-all over NCCL / NVLink), folds them in the visibility order of the slabs
(`vr_sort_groups`, `vr_composite_bricks`) and the finished strips are gathered.

Marshalling and torch.distributed plumbing only: every arithmetic step runs in libvr's kernels.
BASELINE.json's north star for this round is one GPU ("no sharding and no collectives"): this
module is the NEXT-1 row, exercised on one GPU by rendering the slabs one after the other
(tests/test_gpu_sortlast_sharded.py) and, for the exchange, over gloo on CPU.
"""
from __future__ import annotations

import numpy as np

from . import vr


def slab_groups(brick_grid, world: int) -> list:
    """Split the brick grid's z-layers into `world` contiguous slabs, as evenly as possible.
    Returns world + 1 ascending brick ids (group g = bricks [first[g], first[g+1]))."""
    gx, gy, gz = (int(v) for v in brick_grid)
    layer = gx * gy
    cuts = [(gz * g) // world for g in range(world + 1)]
    return [layer * c for c in cuts]


def strip_rows(height: int, world: int) -> int:
    """Rows per strip (the last strips may be padding)."""
    return -(-int(height) // int(world))


class Shard:
    """One rank's share of a sharded sort-last renderer."""

    def __init__(self, ctx: "vr.Context", dims, brick, rank: int, world: int):
        self.ctx, self.rank, self.world = ctx, int(rank), int(world)
        self.dims, self.brick = tuple(dims), tuple(brick)
        grid = [-(-n // min(b, n)) for n, b in zip(dims, brick)]
        self.group_first = slab_groups(grid, world)
        self.first, self.end = self.group_first[rank], self.group_first[rank + 1]
        self.arena = None

    def layout(self):
        """Bytes of this rank's cube and meta buffers."""
        return vr.window_layout(self.dims, self.brick, self.first, self.end)

    def bind(self):
        self.ctx.set_brick_window(self.first, self.end)

    def render_partial(self, torch, mode, W, H, tau=0.99):
        """Premultiplied (C, A) frame (EA) or per-pixel maximum with -inf where nothing was sampled
        (MIP) of the resident bricks under the current view / transfer function."""
        ctx = self.ctx
        ch = 4 if mode == vr.MODE_EA else 1
        out = torch.empty((H, W, ch), dtype=torch.float32, device="cuda")
        ids = ctx.sort_bricks(mode)
        parts, n, nbytes = ctx.partial_layout(mode, ids)
        if self.arena is None or self.arena.numel() < nbytes:
            self.arena = torch.empty(int(nbytes * 1.25) + 256, dtype=torch.uint8, device="cuda")
        vr.Context.bind_partials(parts, n, self.arena)
        ctx.render_bricks(mode, parts, n, tau)
        bg = (0.0, 0.0, 0.0, 0.0) if mode == vr.MODE_EA else (float("-inf"), 0.0, 0.0, 0.0)
        ctx.composite_bricks(mode, parts, n, out, bg)
        return out

    def fold_strip(self, torch, mode, versions, W, H, bg):
        """versions: [world, rows, W, ch] - every rank's version of THIS rank's strip, indexed by
        rank.  Folds them in the slabs' visibility order into rows of a full frame buffer and
        returns the strip [rows, W, ch]."""
        ctx, world = self.ctx, self.world
        rows = versions.shape[1]
        y0 = self.rank * rows
        h = max(0, min(rows, H - y0))
        ch = versions.shape[3]
        frame = torch.empty((H, W, ch), dtype=torch.float32, device=versions.device)
        order = ctx.sort_groups(self.group_first)
        parts = (vr.Partial * world)()
        n = 0
        for g in order:
            if h == 0 or self.group_first[g + 1] == self.group_first[g]:
                continue
            parts[n].brick = self.first            # any resident brick: the id is not used by the fold
            parts[n].x0, parts[n].y0, parts[n].w, parts[n].h = 0, y0, W, h
            parts[n].pitch_px = W
            parts[n].d_data = versions[int(g)].data_ptr()
            n += 1
        ctx.composite_bricks(mode, parts, n, frame, bg)
        out = torch.zeros((rows, W, ch), dtype=torch.float32, device=versions.device)
        out[:h] = frame[y0:y0 + h]
        return out


def exchange_strips(dist, partial, world: int):
    """Direct send: cut `partial` [H, W, ch] into `world` strips of equal rows (zero padded) and
    give strip r of every rank to rank r.  Returns [world, rows, W, ch] indexed by sender."""
    import torch
    H, W, ch = partial.shape
    rows = strip_rows(H, world)
    send = torch.zeros((world * rows, W, ch), dtype=partial.dtype, device=partial.device)
    send[:H] = partial
    if world == 1:
        return send.view(1, rows, W, ch)
    recv = torch.empty_like(send)
    dist.all_to_all_single(recv, send)
    return recv.view(world, rows, W, ch)


def gather_strips(dist, strip, world: int, H: int):
    """All ranks' finished strips -> the frame [H, W, ch] on every rank."""
    import torch
    if world == 1:
        return strip[:H]
    parts = [torch.empty_like(strip) for _ in range(world)]
    dist.all_gather(parts, strip.contiguous())
    return torch.cat(parts, dim=0)[:H]
