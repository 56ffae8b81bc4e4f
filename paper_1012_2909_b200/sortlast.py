"""Sort-last rendering with the bricks sharded over several GPUs.

PAPER.md line 13 (abstract) and line 19 (section 1): the framework renders sub-volumes on
"distributed GPUs" and composites their images.  Here rank r of `world` holds one slab of whole
z-layers of bricks (`vr_set_brick_window`), renders the partial images of its resident bricks and
folds them into ONE premultiplied partial frame (`vr_render_bricks` + `vr_composite_bricks`); the
frame is then cut into `world` strips of rows and rank r finishes strip r.  Two exchanges:

* fused (`PeerFold`, the default on GPUs): ONE kernel per rank (`vr_fold_peers`) reads strip r of every rank's
  partial frame straight from the owners' memory (peer pointers over NVLink, mapped once with CUDA IPC), folds the
  versions in the visibility order of the slabs (`vr_sort_groups`) and stores the finished rows into every rank's
  final frame: exchange, over-operator and gather in one launch, no staging copy, no per-frame allocation;
* staged (`exchange_strips` + `Shard.fold_strip` + `gather_strips`): `all_to_all_single`, a separate fold, `all_gather`
  (what runs over gloo on CPU, and the A/B baseline of the fused path).

Slabs are cut either evenly by brick layers (`slab_groups`) or so that the heaviest slab's projected screen area
over a set of reference views is smallest (`plan_slabs`, `balanced_groups`).

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


def balanced_groups(layer_weights, layer_bricks: int, world: int) -> list:
    """Contiguous partition of the z-layers into `world` slabs minimising the heaviest slab's weight (linear
    partition, dynamic programming; empty slabs allowed only if world exceeds the number of layers).
    Returns world + 1 ascending brick ids like slab_groups."""
    wts = [float(v) for v in layer_weights]
    n = len(wts)
    pre = [0.0]
    for v in wts:
        pre.append(pre[-1] + v)
    INF = float("inf")
    k_max = min(world, n)
    # best[k][i]: smallest possible heaviest slab when the first i layers form k non-empty slabs
    best = [[INF] * (n + 1) for _ in range(k_max + 1)]
    cut = [[0] * (n + 1) for _ in range(k_max + 1)]
    best[0][0] = 0.0
    for k in range(1, k_max + 1):
        for i in range(k, n + 1):
            for j in range(k - 1, i):
                cost = max(best[k - 1][j], pre[i] - pre[j])
                if cost < best[k][i]:
                    best[k][i], cut[k][i] = cost, j
    cuts, i = [n], n
    for k in range(k_max, 0, -1):
        i = cut[k][i]
        cuts.append(i)
    cuts = cuts[::-1] + [n] * (world - k_max)             # surplus ranks get empty slabs
    return [int(layer_bricks) * c for c in cuts]


def plan_slabs(dims, brick, frame, views, step: float, world: int, device: int = 0) -> list:
    """Slabs balanced by projected area: the weight of a z-layer of bricks is the summed area of its bricks' screen
    rectangles (vr_partial_layout, geometry only) averaged over the reference `views` (4x4 matrices)."""
    import torch
    grid = [-(-n // min(b, n)) for n, b in zip(dims, brick)]
    layer = grid[0] * grid[1]
    ctx = vr.Context(device)
    ctx.set_brick_window(0, 0)                              # geometry only: no brick resident
    dummy = torch.zeros(256, dtype=torch.uint8, device="cuda")
    ctx.attach_cube(dims, brick, dummy, dummy)
    ids = np.arange(layer * grid[2], dtype=np.int32)
    W, H = frame
    wts = np.zeros(grid[2])
    for M in views:
        ctx.set_view(M, W, H, step)
        parts, n, _ = ctx.partial_layout(vr.MODE_EA, ids)
        area = np.array([parts[i].w * parts[i].h for i in range(n)], dtype=np.float64)
        wts += area.reshape(grid[2], layer).sum(axis=1)
    ctx.close()
    return balanced_groups(wts / max(1, len(views)), layer, world)


def strip_rows(height: int, world: int) -> int:
    """Rows per strip (the last strips may be padding)."""
    return -(-int(height) // int(world))


class Shard:
    """One rank's share of a sharded sort-last renderer."""

    def __init__(self, ctx: "vr.Context", dims, brick, rank: int, world: int, group_first=None):
        self.ctx, self.rank, self.world = ctx, int(rank), int(world)
        self.dims, self.brick = tuple(dims), tuple(brick)
        grid = [-(-n // min(b, n)) for n, b in zip(dims, brick)]
        self.group_first = list(group_first) if group_first is not None else slab_groups(grid, world)
        self.first, self.end = self.group_first[rank], self.group_first[rank + 1]
        self.arena = None

    def layout(self):
        """Bytes of this rank's cube and meta buffers."""
        return vr.window_layout(self.dims, self.brick, self.first, self.end)

    def bind(self):
        self.ctx.set_brick_window(self.first, self.end)

    def render_partial(self, torch, mode, W, H, tau=0.99, out=None):
        """Premultiplied (C, A) frame (EA) or per-pixel maximum with -inf where nothing was sampled
        (MIP) of the resident bricks under the current view / transfer function (into `out` if given)."""
        ctx = self.ctx
        ch = 4 if mode == vr.MODE_EA else 1
        if out is None:
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


class PeerFold:
    """The fused exchange of one rank: its partial and final frame buffers, every peer's mapped into this process once
    (CUDA IPC handles travel through `dist.all_gather_object`), and per frame one `vr_fold_peers` launch between two
    stream-ordered barriers (tiny all-reduces: plumbing, not data).  `peers` = [(partial_ptr, final_ptr)] lets one process
    stand for all ranks (single-GPU tests: plain pointers, no IPC)."""

    def __init__(self, shard: Shard, torch, mode, W, H, dist=None, peers=None):
        self.shard, self.torch, self.mode, self.dist, self.W, self.H = shard, torch, mode, dist, int(W), int(H)
        ch = 4 if mode == vr.MODE_EA else 1
        self.partial = torch.zeros((H, W, ch), dtype=torch.float32, device="cuda")
        self.final = torch.zeros((H, W, ch), dtype=torch.float32, device="cuda")
        self.rows = strip_rows(H, shard.world)
        self.in_ptrs = self.out_ptrs = None
        if peers is not None:
            self.bind(peers)
        elif dist is not None and shard.world > 1:
            ctx, rank = shard.ctx, shard.rank
            mine = (ctx.ipc_export(self.partial), ctx.ipc_export(self.final))
            everyone = [None] * shard.world
            dist.all_gather_object(everyone, mine)
            self.bind([(self.partial.data_ptr(), self.final.data_ptr()) if r == rank else
                       (ctx.ipc_open(*everyone[r][0]), ctx.ipc_open(*everyone[r][1])) for r in range(shard.world)])
            self.flag = torch.zeros(1, dtype=torch.float32, device="cuda")
        else:
            self.bind([(self.partial.data_ptr(), self.final.data_ptr())])

    def bind(self, peers):
        self.in_ptrs, self.out_ptrs = [p[0] for p in peers], [p[1] for p in peers]

    def barrier(self):
        """Kernels enqueued after it start only when every rank's earlier kernels are done.  NCCL: a one-float
        all-reduce on the stream (no host wait); other backends (gloo in the tests): synchronise, then a host barrier."""
        if self.dist is not None and self.shard.world > 1 and hasattr(self, "flag"):
            if self.dist.get_backend() == "nccl":
                self.dist.all_reduce(self.flag)
            else:
                self.torch.cuda.synchronize()
                self.dist.barrier()

    def render(self, tau=0.99):
        return self.shard.render_partial(self.torch, self.mode, self.W, self.H, tau, out=self.partial)

    def fold(self, bg):
        """This rank's strip of the frame, folded from all ranks' partial frames into all ranks' final frames."""
        sh = self.shard
        y0 = min(self.H, sh.rank * self.rows)
        rows = max(0, min(self.rows, self.H - y0))
        order = sh.ctx.sort_groups(sh.group_first)
        if self.mode != vr.MODE_EA:
            bg = (bg[0], 0.0, 0.0, 0.0)
        sh.ctx.fold_peers(self.mode, self.in_ptrs, order, self.W, self.H, self.W, y0, rows, self.out_ptrs, self.W, bg)

    def frame(self, bg, tau=0.99):
        """One frame: render the slab, barrier, fold + gather over peer memory, barrier."""
        self.render(tau)
        self.barrier()
        self.fold(bg)
        self.barrier()
        return self.final


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
