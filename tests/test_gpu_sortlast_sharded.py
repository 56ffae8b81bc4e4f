"""NEXT-1: bricks sharded over ranks in z-slabs, partial frames folded in the
slabs' visibility order.  One GPU: the ranks' contexts render one after the other (nothing waits
on anything), the exchange is done by slicing.  Reference = the single-context sort-last frame of
the same cube (itself checked against the oracle in test_gpu_parity.py)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def _render_sharded(torch, vr, wl, sl, w, world, mode, M, tf, bg, tau):
    W, H = w.frame
    src = wl.make_sources(w)
    shards, partials = [], []
    for r in range(world):
        ctx = vr.Context(0)
        sh = sl.Shard(ctx, w.dims, w.brick, r, world)
        sh.bind()
        cb, mb = sh.layout()
        d_cube = torch.empty(max(cb // 4, 1), dtype=torch.float32, device="cuda")
        d_meta = torch.empty(max(mb, 1), dtype=torch.uint8, device="cuda")
        ctx.generate_cube(w.seed, w.dims, w.brick, d_cube, d_meta, sources=src, continuum=w.continuum)
        ctx.set_view(M, W, H, w.step)
        ctx.set_transfer_function(*tf)
        partials.append(sh.render_partial(torch, mode, W, H, tau))
        shards.append((sh, d_cube, d_meta))
    rows = sl.strip_rows(H, world)
    strips = []
    for r in range(world):
        versions = torch.stack([_strip(torch, p, r, rows) for p in partials])      # what rank r receives
        strips.append(shards[r][0].fold_strip(torch, mode, versions, W, H, bg))
    torch.cuda.synchronize()
    return torch.cat(strips, dim=0)[:H].cpu().numpy(), [s[0] for s in shards]


def _strip(torch, p, r, rows):
    H, W, ch = p.shape
    out = torch.zeros((rows, W, ch), dtype=p.dtype, device=p.device)
    h = max(0, min(rows, H - r * rows))
    out[:h] = p[r * rows:r * rows + h]
    return out


@pytest.mark.parametrize("world", [2, 3])
@pytest.mark.parametrize("az", [20, 90, 200])
def test_sharded_slabs_equal_single_context(world, az):
    import torch
    from paper_1012_2909_b200 import sortlast as sl, vr, workloads as wl
    import helpers
    w = wl.scaled(wl.C3, "shard", (96, 80, 160), (32, 32, 32), (160, 90), n_sources=40)
    M = wl.perspective_camera(w.dims, w.frame, azimuth_deg=az)
    tf = wl.tf_fog()
    bg = (0.05, 0.1, 0.2, 0.0)
    sc = helpers.Scene(w.dims, w.brick, gen={"seed": w.seed, "sources": wl.make_sources(w), "continuum": w.continuum})
    W, H = w.frame
    ref, _, _ = sc.render_sortlast(M, W, H, w.step, vr.MODE_EA, tf=tf, bg=bg, tau=2.0)
    got, shards = _render_sharded(torch, vr, wl, sl, w, world, vr.MODE_EA, M, tf, bg, 2.0)
    assert np.abs(got - ref).max() <= 2e-6
    assert sum(s.end - s.first for s in shards) == 3 * 3 * 5        # every brick resident on exactly one rank
    ref_m, _, _ = sc.render_sortlast(M, W, H, w.step, vr.MODE_MIP, bg=(-3.0, 0, 0, 0))
    got_m, _ = _render_sharded(torch, vr, wl, sl, w, world, vr.MODE_MIP, M, tf, (-3.0, 0, 0, 0), 2.0)
    assert np.array_equal(got_m[..., 0], ref_m)                       # max is exact in any order


def test_window_refuses_whole_frame_renders_and_foreign_bricks():
    import torch
    from paper_1012_2909_b200 import sortlast as sl, vr, workloads as wl
    w = wl.scaled(wl.C3, "shard", (64, 64, 128), (32, 32, 32), (64, 36), n_sources=4)
    ctx = vr.Context(0)
    sh = sl.Shard(ctx, w.dims, w.brick, 1, 2)
    sh.bind()
    cb, mb = sh.layout()
    full_cb, _ = vr.cube_layout(w.dims, w.brick)
    assert cb * 2 == full_cb
    d_cube = torch.empty(cb // 4, dtype=torch.float32, device="cuda")
    d_meta = torch.empty(mb, dtype=torch.uint8, device="cuda")
    ctx.generate_cube(w.seed, w.dims, w.brick, d_cube, d_meta, sources=wl.make_sources(w))
    ctx.set_view(wl.perspective_camera(w.dims, w.frame), 64, 36, 0.5)
    ctx.set_transfer_function(*wl.tf_fog())
    out = torch.empty((36, 64, 4), dtype=torch.float32, device="cuda")
    with pytest.raises(vr.VRError) as e:
        ctx.render_ea(out)
    assert e.value.status == vr.ERR_STATE
    assert set(ctx.sort_bricks(vr.MODE_MIP)) <= set(range(sh.first, sh.end))
    t = torch.empty(32 ** 3, dtype=torch.float32, device="cuda")
    with pytest.raises(vr.VRError):
        ctx.download_brick(0, t)
    # resident bricks hold the same bytes as in an unsharded context
    ctx.download_brick(sh.first, t)
    full = vr.Context(0)
    fc, fm = vr.cube_layout(w.dims, w.brick)
    dc = torch.empty(fc // 4, dtype=torch.float32, device="cuda")
    dm = torch.empty(fm, dtype=torch.uint8, device="cuda")
    full.generate_cube(w.seed, w.dims, w.brick, dc, dm, sources=wl.make_sources(w))
    t2 = torch.empty(32 ** 3, dtype=torch.float32, device="cuda")
    full.download_brick(sh.first, t2)
    torch.cuda.synchronize()
    assert torch.equal(t, t2)


def test_wallaby_scale_slab_one_rank_of_many():
    """the WALLABY cube, 6144 x 6144 x 16384 (2.25 TiB at 4 bytes, line 13 "2.2
    terabyte"), is what the framework is meant to reach.  One B200 holds one rank's share of it: rank
    20 of a 32-way z-slab split = 2 layers of 24 x 24 bricks of 256^3 (1152 bricks, 77 GB), with GLOBAL
    voxel coordinates up to 16384 and GLOBAL brick ids (23040...) whose occupancy-word offsets pass
    2^32.  Its partial images are compared, on sampled pixels, with the oracle's partial image of the
    same brick (float32 instantiation, bit for bit)."""
    import torch
    from paper_1012_2909_b200 import sortlast as sl, vr, workloads as wl
    from oracle import ovr
    torch.cuda.empty_cache()
    free, _ = torch.cuda.mem_get_info()
    if free < 95e9:
        pytest.skip("needs ~85 GB of free HBM")
    w = wl.scaled(wl.C3, "WALLABY-shaped", (6144, 6144, 16384), (256, 256, 256), (1920, 1080), n_sources=6000)
    assert w.brick_grid == (24, 24, 64)
    world, rank = 32, 20
    ctx = vr.Context(0)
    sh = sl.Shard(ctx, w.dims, w.brick, rank, world)
    assert (sh.first, sh.end) == (24 * 24 * 40, 24 * 24 * 42)
    assert sh.end * 32 * 32 * 32 * 16 > 2 ** 32                 # occupancy words before the slab's last brick
    sh.bind()
    cb, mb = sh.layout()
    d_cube = torch.empty(cb // 4, dtype=torch.float32, device="cuda")
    d_meta = torch.empty(mb, dtype=torch.uint8, device="cuda")
    ctx.generate_cube(w.seed, w.dims, w.brick, d_cube, d_meta, sources=wl.make_sources(w), continuum=w.continuum)
    W, H = w.frame
    M = wl.perspective_camera(w.dims, w.frame, azimuth_deg=35.0)
    tf = wl.tf_src()
    ctx.set_view(M, W, H, w.step)
    ctx.set_transfer_function(*tf)
    for mode, omode in ((vr.MODE_EA, ovr.EA), (vr.MODE_MIP, ovr.MIP)):
        ids = ctx.sort_bricks(mode)
        assert len(ids) > 100 and set(ids) <= set(range(sh.first, sh.end))
        parts, n, nbytes = ctx.partial_layout(mode, ids)
        arena = torch.zeros(nbytes + 256, dtype=torch.uint8, device="cuda")
        offs = [(parts[i].d_data or 0) for i in range(n)]
        vr.Context.bind_partials(parts, n, arena)
        ctx.render_bricks(mode, parts, n, 0.99)
        torch.cuda.synchronize()
        host = arena.cpu().numpy()
        ch = 4 if mode == vr.MODE_EA else 1
        # bricks of the slab's lower layer away from the grid's +x / +y faces: the oracle stores plain bricks
        # (no halo), so it needs the 2 x 2 x 2 neighbourhood, which is resident for these
        ok = [i for i in range(n) if parts[i].brick // 576 == 40 and parts[i].brick % 24 < 23 and (parts[i].brick // 24) % 24 < 23]
        assert len(ok) > 20
        for i in (ok[0], ok[len(ok) // 2], ok[-1]):
            p = parts[i]
            img = host[offs[i]:offs[i] + 4 * ch * p.w * p.h].view(np.float32).reshape(p.h, p.w, ch)
            bricks = {}
            for dz in (0, 1):
                for dy in (0, 1):
                    for dx in (0, 1):
                        nbid = int(p.brick) + dx + 24 * dy + 576 * dz
                        t = torch.empty(256 ** 3, dtype=torch.float32, device="cuda")
                        ctx.download_brick(nbid, t)
                        bricks[nbid] = t.cpu().numpy().reshape(256, 256, 256)
                        del t
            vol = ovr.Volume(w.dims, w.brick, bricks)
            bw, bh = min(6, p.w), min(6, p.h)
            rx, ry = p.x0 + (p.w - bw) // 2, p.y0 + (p.h - bh) // 2
            want = ovr.render_brick(vol, M, W, H, w.step, omode, int(p.brick), (rx, ry, bw, bh), w.brick,
                                    precision=ovr.F32, tf=tf, tau=0.99)
            got = img[ry - p.y0:ry - p.y0 + bh, rx - p.x0:rx - p.x0 + bw]
            got = got if ch == 4 else got[..., 0]
            assert np.isfinite(want).any()
            assert np.array_equal(got, want), (mode, int(p.brick))
    part = sh.render_partial(torch, vr.MODE_EA, W, H, 0.99)
    torch.cuda.synchronize()
    assert float(part[..., 3].max()) <= 1.0 + 1e-6 and float(part[..., 3].min()) >= 0.0


def _oracle_two_level(ovr, vol, M, W, H, step, omode, brick, grid, group_first, tf, tau, bg, miss):
    """The sharded frame by the oracle's own pieces, float32: per-brick partial images (O-8 SORT-LAST), folded per
    slab in the bricks' visibility order without a background, then the slabs' images folded in the slabs' order."""
    keys, _ = ovr.visibility_keys(M, W, H, step, brick, grid)
    order = ovr.visibility_order(keys)
    full = (0, 0, W, H)
    slab_imgs, slab_keys = [], []
    for g in range(len(group_first) - 1):
        ids = [int(b) for b in order if group_first[g] <= b < group_first[g + 1]]
        imgs = [ovr.render_brick(vol, M, W, H, step, omode, b, full, brick, ovr.F32, tf=tf, tau=tau) for b in ids]
        if omode == ovr.EA:
            img = ovr.composite(omode, [full] * len(ids), imgs, None, W, H, bg=(0, 0, 0, 0), precision=ovr.F32) if ids else np.zeros((H, W, 4), np.float32)
        else:
            img = np.max(np.stack(imgs), axis=0) if ids else np.full((H, W), -np.inf, np.float32)
        slab_imgs.append(img)
        slab_keys.append(min(keys[group_first[g]:group_first[g + 1]]) if ids else np.iinfo(np.int32).max)
    slab_order = np.argsort(np.array(slab_keys), kind="stable").astype(np.int32)
    return ovr.composite(omode, [full] * len(slab_imgs), slab_imgs, slab_order, W, H, bg=bg, miss=miss, precision=ovr.F32)


@pytest.mark.parametrize("world,balanced", [(2, False), (3, True), (7, False)])
def test_fused_peer_fold_equals_the_oracle(world, balanced):
    """NEXT-1: one vr_fold_peers launch per rank (exchange + fold + gather through the peers' pointers; here all
    ranks live in one process on one device, so the pointers are plain) against the ORACLE's sort-last pieces put
    together slab by slab.  world = 7 exceeds the 5 brick layers: two ranks hold empty slabs."""
    import torch
    from paper_1012_2909_b200 import sortlast as sl, vr, workloads as wl
    from oracle import ovr
    import helpers
    w = wl.scaled(wl.C3, "shard", (96, 80, 160), (32, 32, 32), (160, 90), n_sources=40)
    W, H = w.frame
    src = wl.make_sources(w)
    tf = wl.tf_fog()
    bg = (0.05, 0.1, 0.2, 0.3)
    grid = w.brick_grid
    M0 = wl.perspective_camera(w.dims, w.frame, azimuth_deg=20.0)
    group_first = sl.plan_slabs(w.dims, w.brick, w.frame, [wl.perspective_camera(w.dims, w.frame, azimuth_deg=a) for a in (0, 120, 240)],
                                w.step, world) if balanced else None
    sc = helpers.Scene(w.dims, w.brick, gen={"seed": w.seed, "sources": src, "continuum": w.continuum})
    vol = sc.oracle_volume()
    for mode, omode, tau in ((vr.MODE_EA, ovr.EA, 0.95), (vr.MODE_MIP, ovr.MIP, 2.0)):
        shards, folds, keep = [], [], []
        for r in range(world):
            ctx = vr.Context(0)
            sh = sl.Shard(ctx, w.dims, w.brick, r, world, group_first=group_first)
            sh.bind()
            cb, mb = sh.layout()
            d_cube = torch.empty(max(cb // 4, 64), dtype=torch.float32, device="cuda")
            d_meta = torch.empty(max(mb, 256), dtype=torch.uint8, device="cuda")
            ctx.generate_cube(w.seed, w.dims, w.brick, d_cube, d_meta, sources=src, continuum=w.continuum)
            ctx.set_transfer_function(*tf)
            shards.append(sh)
            keep.append((d_cube, d_meta))
            folds.append(sl.PeerFold(sh, torch, mode, W, H))
        peers = [(f.partial.data_ptr(), f.final.data_ptr()) for f in folds]
        for f in folds:
            f.bind(peers)
        assert sum(s.end - s.first for s in shards) == grid[0] * grid[1] * grid[2]
        for az in (20.0, 200.0):
            M = wl.perspective_camera(w.dims, w.frame, azimuth_deg=az)
            for f in folds:
                f.shard.ctx.set_view(M, W, H, w.step)
                f.render(tau)
            torch.cuda.synchronize()                                  # the barrier of the multi-process path
            for f in folds:
                f.fold(bg if mode == vr.MODE_EA else (-3.0, 0, 0, 0))
            torch.cuda.synchronize()
            want = _oracle_two_level(ovr, vol, M, W, H, w.step, omode, w.brick, grid, shards[0].group_first, tf, tau, bg, -3.0)
            for f in folds:                                           # every rank holds the whole finished frame
                got = f.final.cpu().numpy()
                got = got if mode == vr.MODE_EA else got[..., 0]
                assert np.array_equal(got, want), (world, mode, az, f.shard.rank)
    del M0


def _ipc_worker(rank, world, port, out_dir):
    """One rank of the multi-process path: its own CUDA context on the one device, the peers' frames mapped with CUDA
    IPC (vr_ipc_export / vr_ipc_open), vr_fold_peers reading and writing through the mapped pointers."""
    import os
    import numpy as np
    import torch
    import torch.distributed as dist
    from paper_1012_2909_b200 import sortlast as sl, vr, workloads as wl
    os.environ["MASTER_ADDR"], os.environ["MASTER_PORT"] = "127.0.0.1", str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    torch.cuda.set_device(0)
    w = wl.scaled(wl.C3, "shard", (96, 80, 160), (32, 32, 32), (160, 90), n_sources=40)
    W, H = w.frame
    ctx = vr.Context(0)
    sh = sl.Shard(ctx, w.dims, w.brick, rank, world)
    sh.bind()
    cb, mb = sh.layout()
    d_cube = torch.empty(max(cb // 4, 64), dtype=torch.float32, device="cuda")
    d_meta = torch.empty(max(mb, 256), dtype=torch.uint8, device="cuda")
    ctx.generate_cube(w.seed, w.dims, w.brick, d_cube, d_meta, sources=wl.make_sources(w), continuum=w.continuum)
    ctx.set_transfer_function(*wl.tf_fog())
    pf = sl.PeerFold(sh, torch, vr.MODE_EA, W, H, dist=dist)
    assert len(pf.in_ptrs) == world and pf.in_ptrs[rank] == pf.partial.data_ptr()
    frames = []
    for az in (20.0, 200.0):
        ctx.set_view(wl.perspective_camera(w.dims, w.frame, azimuth_deg=az), W, H, w.step)
        frames.append(pf.frame((0.05, 0.1, 0.2, 0.3), tau=0.95).clone())
    torch.cuda.synchronize()
    np.save(os.path.join(out_dir, f"rank{rank}.npy"), torch.stack(frames).cpu().numpy())
    dist.barrier()
    dist.destroy_process_group()


def test_fused_fold_across_two_processes_over_cuda_ipc(tmp_path):
    """The multi-process form of NEXT-1 on the one GPU this run has: two processes, each holding a slab, exchange
    CUDA IPC handles over gloo; every rank's kernel reads the other's partial frame and writes the other's final frame
    through the mapped pointers.  No kernel waits on another (host barriers only).  Both ranks must end with the frame
    the oracle's pieces give."""
    import socket
    import torch
    import torch.multiprocessing as mp
    from paper_1012_2909_b200 import sortlast as sl, vr, workloads as wl
    from oracle import ovr
    import helpers
    with socket.socket() as sck:
        sck.bind(("127.0.0.1", 0))
        port = sck.getsockname()[1]
    ctx = mp.get_context("spawn")
    procs = [ctx.Process(target=_ipc_worker, args=(r, 2, port, str(tmp_path))) for r in range(2)]
    for p in procs:
        p.start()
    for p in procs:
        p.join(timeout=600)
        assert p.exitcode == 0, "a rank failed or hung"
    w = wl.scaled(wl.C3, "shard", (96, 80, 160), (32, 32, 32), (160, 90), n_sources=40)
    W, H = w.frame
    sc = helpers.Scene(w.dims, w.brick, gen={"seed": w.seed, "sources": wl.make_sources(w), "continuum": w.continuum})
    vol = sc.oracle_volume()
    group_first = sl.slab_groups(w.brick_grid, 2)
    got = [np.load(tmp_path / f"rank{r}.npy") for r in range(2)]
    assert np.array_equal(got[0], got[1])
    for i, az in enumerate((20.0, 200.0)):
        M = wl.perspective_camera(w.dims, w.frame, azimuth_deg=az)
        want = _oracle_two_level(ovr, vol, M, W, H, w.step, ovr.EA, w.brick, w.brick_grid, group_first, wl.tf_fog(), 0.95,
                                 (0.05, 0.1, 0.2, 0.3), 0.0)
        assert np.array_equal(got[0][i], want), az
