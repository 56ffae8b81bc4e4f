"""vr_composite_bricks_static: the sort-last fold for callers that must not allocate.  Its
descriptor scratch is a static __device__ array of the library instead of a cudaMalloc'd buffer; the frames must
equal vr_composite_bricks' bit for bit (the tolerance of the parity tests for the float32 reading is equality), on
two calls in a row that share the array, and through them the oracle's sort-last frame.

Collected last on purpose (the file name): the suite runs with pytest -x.  Runs alone in a fresh process and
after the other tests alike: it builds its own context and touches nothing the others leave behind."""
import numpy as np
import pytest

from paper_1012_2909_b200 import workloads as wl

pytestmark = pytest.mark.gpu

BG = (0.25, 0.5, 0.125, 0.75)


@pytest.fixture(scope="module")
def H():
    import helpers
    helpers.torch_cuda()
    helpers.FORCED_OPTIONS.clear()
    return helpers


def _partials(sc, torch, mode, M, W, Hh, step, tf, tau):
    """Per-brick partial images of one view through the existing calls; returns (parts, n, arena)."""
    ctx = sc.ctx
    ctx.set_view(M, W, Hh, step)
    if tf is not None:
        ctx.set_transfer_function(*tf)
    ids = ctx.sort_bricks(mode)
    parts, n, nbytes = ctx.partial_layout(mode, ids)
    arena = torch.zeros(max(nbytes, 256), dtype=torch.uint8, device="cuda")
    sc.vr.Context.bind_partials(parts, n, arena)
    ctx.render_bricks(mode, parts, n, tau)
    return parts, n, arena


def test_static_composite_equals_the_allocating_path_on_two_calls_in_a_row(H):
    import torch
    from oracle import ovr
    w = wl.scaled(wl.C2, "noalloc", (96, 80, 128), (32, 32, 32), (160, 90), n_sources=8)
    sc = H.Scene(w.dims, w.brick, gen={"seed": w.seed, "sources": wl.make_sources(w)})
    vr = sc.vr
    W, Hh = w.frame
    tf = wl.tf_fog()
    # call 1: emission-absorption, every brick of the view (the longer list); call 2: MIP of another view and, last,
    # a SHORTER emission-absorption list, so that entries of the earlier calls are still in the array beyond n
    cases = [(vr.MODE_EA, 30.0, tf, 0.99, BG, None), (vr.MODE_MIP, 200.0, None, 2.0, (-3.0, 0.0, 0.0, 0.0), None),
             (vr.MODE_EA, 200.0, tf, 0.99, BG, 5)]
    for mode, az, table, tau, bg, keep in cases:
        M = wl.perspective_camera(w.dims, w.frame, azimuth_deg=az)
        parts, n, arena = _partials(sc, torch, mode, M, W, Hh, w.step, table, tau)
        n = n if keep is None else min(n, keep)
        ch = 4 if mode == vr.MODE_EA else 1
        want = torch.full((Hh, W, ch), -7.0, dtype=torch.float32, device="cuda")
        got = torch.full((Hh, W, ch), 7.0, dtype=torch.float32, device="cuda")
        sc.ctx.composite_bricks(mode, parts, n, want, bg)
        sc.ctx.composite_bricks_static(mode, parts, n, got, bg)
        torch.cuda.synchronize()
        assert torch.equal(got, want), (mode, az, keep)
        got.fill_(7.0)
        free_before, _ = torch.cuda.mem_get_info()                       # (the first call ever loads the kernel's module)
        sc.ctx.composite_bricks_static(mode, parts, n, got, bg)          # and again: same array, same answer
        torch.cuda.synchronize()
        free_after, _ = torch.cuda.mem_get_info()
        assert free_after == free_before                                 # no device memory was taken
        assert torch.equal(got, want), (mode, az, keep)
        if keep is None:                                                 # the whole list: the oracle's sort-last frame too
            vol = sc.oracle_volume()
            omode = ovr.EA if mode == vr.MODE_EA else ovr.MIP
            if mode == vr.MODE_EA:
                ref, _, _ = ovr.render(vol, M, W, Hh, w.step, omode, ovr.F32, tf=table, bg=bg, tau=tau,
                                       split=ovr.SPLIT_SORTLAST, partition=w.brick)
            else:                                                        # the maximum is the same however the cube is split
                ref, _, _ = ovr.render(vol, M, W, Hh, w.step, omode, ovr.F32, miss=bg[0])
            g = got.cpu().numpy()
            assert np.array_equal(g if mode == vr.MODE_EA else g[..., 0], ref)
        del arena


def test_static_composite_refuses_more_than_its_maximum(H):
    import torch
    dims, brick = (32, 32, 32), (16, 16, 16)
    cube = np.random.default_rng(2).normal(size=dims[::-1]).astype(np.float32)
    sc = H.Scene(dims, brick, cube=cube)
    vr = sc.vr
    W, Hh = 48, 40
    sc.ctx.set_view(wl.perspective_camera(dims, (W, Hh)), W, Hh, 0.5)
    sc.ctx.set_transfer_function(*wl.tf_fog())
    n = vr.STATIC_MAX_PARTIALS + 1
    img = torch.zeros((Hh, W, 4), dtype=torch.float32, device="cuda")
    out = torch.full((Hh, W, 4), 3.0, dtype=torch.float32, device="cuda")
    parts = (vr.Partial * n)()
    for i in range(n):
        parts[i].brick, parts[i].x0, parts[i].y0, parts[i].w, parts[i].h = 0, 0, 0, W, Hh
        parts[i].pitch_px, parts[i].d_data = W, img.data_ptr()
    with pytest.raises(vr.VRError) as err:
        sc.ctx.composite_bricks_static(vr.MODE_EA, parts, n, out, BG)
    assert err.value.status == vr.ERR_BUFFER and "static maximum of 4096" in str(err.value)
    torch.cuda.synchronize()
    assert bool((out == 3.0).all())                                      # nothing was launched
    # exactly the maximum is served: 4096 transparent images over the background give the background
    sc.ctx.composite_bricks_static(vr.MODE_EA, parts, n - 1, out, BG)
    torch.cuda.synchronize()
    assert torch.equal(out, torch.tensor(BG, dtype=torch.float32, device="cuda").expand(Hh, W, 4))
