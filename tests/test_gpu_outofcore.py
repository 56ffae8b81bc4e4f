"""GPU tests of the out-of-core path (cubes "larger than a single machine
memory limit"): a cube kept brick-major in pinned host memory and streamed slab by slab through a pool of device
slots smaller than the cube (paper_1012_2909_b200/outofcore.py) renders the frame of the oracle's two-level sort-last
composite (per-brick partial images folded per slab, then the slabs folded in their visibility order), bit for bit."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def _scene():
    from paper_1012_2909_b200 import workloads as wl
    w = wl.scaled(wl.C3, "ooc", (96, 80, 160), (32, 32, 32), (160, 90), n_sources=40)
    return w, wl.make_sources(w)


@pytest.mark.parametrize("n_slots", [1, 2, 5])
def test_streamed_cube_equals_the_oracle(n_slots):
    import torch
    from paper_1012_2909_b200 import outofcore, vr, workloads as wl
    from oracle import ovr
    import helpers
    from test_gpu_sortlast_sharded import _oracle_two_level
    helpers.torch_cuda()
    w, src = _scene()
    W, H = w.frame
    sc = helpers.Scene(w.dims, w.brick, gen={"seed": w.seed, "sources": src, "continuum": w.continuum})
    vol = sc.oracle_volume()
    cube = outofcore.StreamedCube(w.dims, w.brick, n_slabs=5, n_slots=n_slots)
    assert cube.n_slabs == 5 and cube.n_slots == n_slots
    cube.ingest_generated(w.seed, sources=src, continuum=w.continuum)
    cb, _ = vr.cube_layout(w.dims, w.brick)
    assert cube.host_bytes() >= cb                                    # the whole cube sits on the host ...
    pool = sum(s["d_cube"].numel() * 4 for s in cube.slots)
    assert n_slots == 5 or pool < cb                                  # ... and the device pool holds a part of it
    bg = (0.05, 0.1, 0.2, 0.3)
    for mode, omode, tau, tf in ((vr.MODE_EA, ovr.EA, 0.95, wl.tf_fog()), (vr.MODE_EA, ovr.EA, 0.99, wl.tf_src()),
                                 (vr.MODE_MIP, ovr.MIP, 2.0, wl.tf_src())):
        cube.set_transfer_function(*tf)
        for az in (20.0, 200.0, 200.0):
            M = wl.perspective_camera(w.dims, w.frame, azimuth_deg=az)
            before = dict(cube.stats)
            got = cube.render(mode, M, W, H, w.step, bg=bg if mode == vr.MODE_EA else (-3.0, 0, 0, 0), tau=tau)
            torch.cuda.synchronize()
            got = got.cpu().numpy()
            got = got if mode == vr.MODE_EA else got[..., 0]
            want = _oracle_two_level(ovr, vol, M, W, H, w.step, omode, w.brick, w.brick_grid, cube.group_first, tf, tau, bg, -3.0)
            assert np.array_equal(got, want), (n_slots, mode, az)
            copied = cube.stats["slabs_copied"] - before["slabs_copied"]
            rendered = cube.stats["slabs_rendered"] - before["slabs_rendered"]
            assert rendered == 5
            if n_slots == 1:
                assert copied >= 4                                    # every slab but (at most) the resident one travels
    if n_slots == 5:
        assert cube.stats["slabs_copied"] <= 5                        # everything fits: each slab travels at most once
    cube.close()


def test_streamed_host_cube_and_view_that_misses():
    """A linear host cube (numpy) ingested slab by slab; a view that looks away renders the background."""
    import torch
    from paper_1012_2909_b200 import outofcore, vr, workloads as wl
    from oracle import ovr
    import helpers
    from test_gpu_sortlast_sharded import _oracle_two_level
    helpers.torch_cuda()
    dims, brick, (W, H) = (50, 37, 61), (16, 16, 16), (64, 48)
    rng = np.random.default_rng(5)
    data = (rng.normal(size=dims[::-1]) * 6.0 + 4.0).astype(np.float32)
    cube = outofcore.StreamedCube(dims, brick, n_slabs=3, n_slots=2)
    cube.ingest_host(data)
    sc = helpers.Scene(dims, brick, cube=data)
    vol = sc.oracle_volume()
    tf = wl.tf_fog()
    cube.set_transfer_function(*tf)
    bg = (0.25, 0.5, 0.125, 0.75)
    M = wl.perspective_camera(dims, (W, H), azimuth_deg=75.0)
    got = cube.render(vr.MODE_EA, M, W, H, 0.5, bg=bg, tau=0.99).cpu().numpy()
    grid = tuple(-(-n // b) for n, b in zip(dims, brick))
    want = _oracle_two_level(ovr, vol, M, W, H, 0.5, ovr.EA, brick, grid, cube.group_first, tf, 0.99, bg, 0.0)
    assert np.array_equal(got, want)
    eye = np.array([25.0, 18.0, -80.0])
    V = wl._look_at(eye, eye + np.array([0.0, 0.0, -1.0]), np.array([0.0, 1.0, 0.0]))
    Maway = (wl._frustum(-0.5, 0.5, -0.4, 0.4, 1.0, 300.0) @ V).astype(np.float32)
    got = cube.render(vr.MODE_EA, Maway, W, H, 0.5, bg=bg, tau=0.99).cpu().numpy()
    assert np.array_equal(got, np.broadcast_to(np.array(bg, dtype=np.float32), got.shape))
    torch.cuda.synchronize()
    cube.close()


def test_streamed_float16_cube_equals_the_oracle_on_the_dequantised_cube():
    """Both halves of NEXT-4 together (O-16 + O-17): a cube stored as float16, kept in pinned host memory and
    streamed through 2 of 5 slots, renders the oracle's two-level composite of the DEquantised cube, bit for bit."""
    import torch
    from paper_1012_2909_b200 import outofcore, vr, workloads as wl
    from oracle import ovr
    import helpers
    from test_gpu_sortlast_sharded import _oracle_two_level
    helpers.torch_cuda()
    w, src = _scene()
    W, H = w.frame
    helpers.FORCED_OPTIONS.clear()
    helpers.FORCED_OPTIONS[vr.OPT_VOXEL_TYPE] = vr.VOXEL_F16
    try:
        sc = helpers.Scene(w.dims, w.brick, gen={"seed": w.seed, "sources": src, "continuum": w.continuum})
    finally:
        helpers.FORCED_OPTIONS.clear()
    vol = sc.oracle_volume()                                          # the values the device holds: float32(float16(v))
    cube = outofcore.StreamedCube(w.dims, w.brick, n_slabs=5, n_slots=2, voxel_type=vr.VOXEL_F16)
    cube.ingest_generated(w.seed, sources=src, continuum=w.continuum)
    cb32, _ = vr.cube_layout_typed(w.dims, w.brick, vr.VOXEL_F32)
    assert cube.host_bytes() < 0.6 * cb32                             # half the bytes on the host, too
    bg = (0.05, 0.1, 0.2, 0.3)
    for mode, omode, tau, tf in ((vr.MODE_EA, ovr.EA, 0.95, wl.tf_fog()), (vr.MODE_EA, ovr.EA, 0.99, wl.tf_src()),
                                 (vr.MODE_MIP, ovr.MIP, 2.0, wl.tf_src())):
        cube.set_transfer_function(*tf)
        M = wl.perspective_camera(w.dims, w.frame, azimuth_deg=140.0)
        got = cube.render(mode, M, W, H, w.step, bg=bg if mode == vr.MODE_EA else (-3.0, 0, 0, 0), tau=tau)
        torch.cuda.synchronize()
        got = got.cpu().numpy()
        got = got if mode == vr.MODE_EA else got[..., 0]
        want = _oracle_two_level(ovr, vol, M, W, H, w.step, omode, w.brick, w.brick_grid, cube.group_first, tf, tau, bg, -3.0)
        assert np.array_equal(got, want), mode
    cube.close()
