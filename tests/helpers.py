"""Shared helpers of the GPU parity tests: build a context from a numpy cube or the device
generator, fetch the cube bytes back for the oracle, compare frames with BASELINE.json's
tolerances (max-abs <= 1e-4, RMS <= 1e-5 per channel in [0,1]; SURVEY.md 8(c) O-12 knife-edge
rule for the flagged pixels)."""
import math

import numpy as np

TOL_MAX, TOL_RMS = 1e-4, 1e-5

# Options every Scene applies to its context (set by the `marcher` fixture of the GPU tests so that
# each marcher variant / skipping level is checked, not only the one the library would pick).
FORCED_OPTIONS = {}


def torch_cuda():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    return torch


class Scene:
    """A cube resident on the GPU through libvr plus the same bytes for the oracle."""

    def __init__(self, dims, brick, cube=None, gen=None):
        torch = torch_cuda()
        from paper_1012_2909_b200 import vr
        from oracle import ovr
        self.vr, self.ovr, self.torch = vr, ovr, torch
        self.dims, self.brick = tuple(dims), tuple(brick)
        cb, mb = vr.cube_layout(dims, brick)
        self.d_cube = torch.empty(cb // 4, dtype=torch.float32, device="cuda")
        self.d_meta = torch.empty(mb, dtype=torch.uint8, device="cuda")
        self.ctx = vr.Context(0)
        for opt, value in FORCED_OPTIONS.items():
            self.ctx.set_option(opt, value)
        if cube is not None:
            self.ctx.upload_cube(np.ascontiguousarray(cube, dtype=np.float32), dims, brick, self.d_cube, self.d_meta)
        else:
            self.ctx.generate_cube(gen["seed"], dims, brick, self.d_cube, self.d_meta, sources=gen.get("sources"),
                                   zero_boxes=gen.get("zero_boxes"), continuum=gen.get("continuum", 0.0))
        self._host = None

    def grid(self):
        return tuple(-(-n // min(b, n)) for n, b in zip(self.dims, self.brick))

    def brick_extent(self, bid):
        g = self.grid()
        bi = (bid % g[0], (bid // g[0]) % g[1], bid // (g[0] * g[1]))
        return tuple(min(min(b, n), n - i * min(b, n)) for i, b, n in zip(bi, self.brick, self.dims)), bi

    def download_brick(self, bid):
        (ex, ey, ez), _ = self.brick_extent(bid)
        t = self.torch.empty(ex * ey * ez, dtype=self.torch.float32, device="cuda")
        self.ctx.download_brick(bid, t)
        self.torch.cuda.synchronize()
        return t.cpu().numpy().reshape(ez, ey, ex)

    def host_cube(self):
        """The cube bytes as they sit on the device, linear [nz, ny, nx]."""
        if self._host is None:
            nx, ny, nz = self.dims
            out = np.zeros((nz, ny, nx), dtype=np.float32)
            g = self.grid()
            B = tuple(min(b, n) for b, n in zip(self.brick, self.dims))
            for bid in range(g[0] * g[1] * g[2]):
                (ex, ey, ez), bi = self.brick_extent(bid)
                x0, y0, z0 = bi[0] * B[0], bi[1] * B[1], bi[2] * B[2]
                out[z0:z0 + ez, y0:y0 + ey, x0:x0 + ex] = self.download_brick(bid)
            self._host = out
        return self._host

    def oracle_volume(self):
        return self.ovr.Volume.linear(self.host_cube())

    # ---- GPU renders, returned as numpy
    def render_ea(self, M, W, H, step, tf, bg=(0, 0, 0, 0), tau=0.99):
        t = self.torch
        self.ctx.set_view(M, W, H, step)
        self.ctx.set_transfer_function(*tf)
        out = t.full((H, W, 4), -7.0, dtype=t.float32, device="cuda")
        self.ctx.render_ea(out, bg, tau)
        t.cuda.synchronize()
        return out.cpu().numpy()

    def render_mip(self, M, W, H, step, miss=0.0, tf=None):
        t = self.torch
        self.ctx.set_view(M, W, H, step)
        out = t.full((H, W), -7.0, dtype=t.float32, device="cuda")
        rgba = None
        if tf is not None:
            self.ctx.set_transfer_function(*tf)
            rgba = t.full((H, W, 4), -7.0, dtype=t.float32, device="cuda")
        self.ctx.render_mip(out, rgba, miss)
        t.cuda.synchronize()
        return out.cpu().numpy() if rgba is None else (out.cpu().numpy(), rgba.cpu().numpy())

    def render_sortlast(self, M, W, H, step, mode, tf=None, bg=(0, 0, 0, 0), tau=0.99, order=None):
        """sort_bricks -> partial_layout -> render_bricks -> composite_bricks.  Returns
        (frame, partial descriptors as python dicts with their images)."""
        t, vr = self.torch, self.vr
        self.ctx.set_view(M, W, H, step)
        if tf is not None:
            self.ctx.set_transfer_function(*tf)
        ids = self.ctx.sort_bricks(mode) if order is None else np.asarray(order, dtype=np.int32)
        parts, n, nbytes = self.ctx.partial_layout(mode, ids)
        arena = t.zeros(max(nbytes, 16), dtype=t.uint8, device="cuda")
        offs = [(parts[i].d_data or 0) for i in range(n)]
        vr.Context.bind_partials(parts, n, arena)
        self.ctx.render_bricks(mode, parts, n, tau)
        ch = 4 if mode == vr.MODE_EA else 1
        out = t.full((H, W, ch), -7.0, dtype=t.float32, device="cuda")
        self.ctx.composite_bricks(mode, parts, n, out, bg)
        t.cuda.synchronize()
        host = arena.cpu().numpy()
        imgs = []
        for i in range(n):
            p = parts[i]
            a = host[offs[i]:offs[i] + 4 * ch * p.w * p.h].view(np.float32).reshape(p.h, p.w, ch)
            imgs.append({"brick": p.brick, "rect": (p.x0, p.y0, p.w, p.h), "image": a if ch == 4 else a[..., 0]})
        frame = out.cpu().numpy()
        return (frame if ch == 4 else frame[..., 0]), imgs, ids


def compare(gpu, o64, flags, o32=None, mode_mip=False, vmin=0.0, vmax=1.0, miss=None, what=""):
    """BASELINE.json tolerances against the fp64 oracle on unflagged pixels; flagged pixels (O-12)
    must match the float32 oracle; flagged fraction < 1 %.  Returns the stats."""
    g, r = gpu.astype(np.float64), o64.astype(np.float64)
    if mode_mip:
        hit = r != miss if miss is not None else np.ones(r.shape, bool)
        unflagged = flags == 0                                # a flagged pixel may legitimately take / miss its only sample
        assert np.array_equal((gpu == miss)[unflagged], (o64 == miss)[unflagged]), f"{what}: miss masks differ"
        g = np.where(hit, (g - vmin) / (vmax - vmin), 0.0)
        r = np.where(hit, (r - vmin) / (vmax - vmin), 0.0)
        g, r = g[..., None], r[..., None]
    ok = flags == 0
    frac = 1.0 - ok.mean()
    assert frac < 0.01, f"{what}: {frac:.4f} of the pixels are knife-edge flagged"
    err = np.abs(g - r)[ok]
    mx = err.max(axis=0) if err.size else np.zeros(g.shape[-1])
    rms = np.sqrt((err ** 2).mean(axis=0)) if err.size else np.zeros(g.shape[-1])
    assert (mx <= TOL_MAX).all(), f"{what}: max abs error {mx} > {TOL_MAX}"
    assert (rms <= TOL_RMS).all(), f"{what}: RMS error {rms} > {TOL_RMS}"
    if o32 is not None and (~ok).any():
        e32 = np.abs(gpu.astype(np.float64) - o32.astype(np.float64))[~ok]
        scale = (vmax - vmin) if mode_mip else 1.0
        assert (e32 / scale <= TOL_MAX).all(), f"{what}: flagged pixels differ from the float32 oracle"
    return {"max": mx, "rms": rms, "flagged": frac}
