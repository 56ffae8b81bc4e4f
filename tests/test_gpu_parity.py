"""GPU parity tests: the CUDA path (through the C ABI, via the thin binding) against the CPU oracle
on the same seeded inputs, element by element.  Tolerances are BASELINE.json's: max-abs <= 1e-4 and
RMS <= 1e-5 per RGBA channel in [0,1] against the fp64 oracle (MIP after normalising by
(m - vmin) / (vmax - vmin)), bit-exact for MIP under axis-aligned orthographic views.  Beyond
that, the kernels implement the canonical float32 arithmetic of SURVEY.md 8(c) O-11, so frames
are also compared bit-for-bit with the float32 instantiation of the oracle.
"""
import math

import numpy as np
import pytest

from paper_1012_2909_b200 import workloads as wl

pytestmark = pytest.mark.gpu

BG = (0.25, 0.5, 0.125, 0.75)


@pytest.fixture(scope="module")
def H():
    import helpers
    helpers.torch_cuda()
    return helpers


# Every test below runs once with the library's own choice of marcher variant and macro-cell
# skipping ("auto") and once per forced variant (0 / 1: ray per thread, CTA per pixel tile / per
# (brick, tile); 3: lockstep ray per warp, folding
# emission-absorption samples in the owning lane "v3s" or through shared memory "v3d", or testing
# every sample against the occupancy bits first "v3o", or with the gathers in a register ring "v3r"; 4: the occupancy marcher for
# dense rays, macro-cell runs first "v4o"; "v3t": the per-brick MIP images in object order), with the macro-cell level of the skipping forced on.
@pytest.fixture(autouse=True, params=["auto", "v0", "v1", "v3s", "v3d", "v3o", "v3r", "v4o", "v3t"])
def marcher(request, H):
    from paper_1012_2909_b200 import vr
    H.FORCED_OPTIONS.clear()
    if request.param != "auto":
        H.FORCED_OPTIONS.update({vr.OPT_VARIANT: int(request.param[1]), vr.OPT_CELL_SKIP: 1})
        if request.param[2:]:
            H.FORCED_OPTIONS[vr.OPT_DENSE] = int(request.param[2] == "d")
            H.FORCED_OPTIONS[vr.OPT_OCCUPANCY] = int(request.param[2] == "o")
            H.FORCED_OPTIONS[vr.OPT_RING] = int(request.param[2] == "r")     # "v3r": sparse fold, gathers through registers
            H.FORCED_OPTIONS[vr.OPT_MIP_TILES] = int(request.param[2] == "t")  # "v3t": per-brick MIP in object order (vr_mip_tiles.cu); else off
    yield request.param
    H.FORCED_OPTIONS.clear()


def noise_cube(shape, seed=0, scale=1.0):
    return (np.random.default_rng(seed).normal(size=shape) * scale).astype(np.float32)


def bit_fraction(a, b):
    return float(np.mean(a.view(np.uint32) == b.view(np.uint32)))


# ------------------------------------------------------------------------------ S0
@pytest.mark.parametrize("dims,brick", [((37, 29, 41), (16, 16, 16)), ((64, 64, 64), (64, 64, 64)),
                                        ((50, 33, 20), (24, 20, 32)), ((8, 8, 8), (16, 16, 16))])
def test_upload_roundtrip_ragged_bricks(H, dims, brick):
    cube = noise_cube(dims[::-1], 1)
    sc = H.Scene(dims, brick, cube=cube)
    assert np.array_equal(sc.host_cube(), cube)
    # device-resident source gives the same bricks
    import torch
    sc2 = H.Scene.__new__(H.Scene)
    sc2.__dict__.update(sc.__dict__)
    d_src = torch.from_numpy(cube).cuda()
    cb, mb = sc.vr.cube_layout(dims, brick)
    sc2.d_cube = torch.empty(cb // 4, dtype=torch.float32, device="cuda")
    sc2.d_meta = torch.empty(mb, dtype=torch.uint8, device="cuda")
    sc2.ctx = sc.vr.Context(0)
    sc2.ctx.upload_cube(d_src, dims, brick, sc2.d_cube, sc2.d_meta)
    sc2._host = None
    assert np.array_equal(sc2.host_cube(), cube)


def test_generator_matches_oracle_and_ignores_brick_size(H):
    w = wl.scaled(wl.C3, "gen", (96, 80, 128), (32, 32, 32), (64, 64), n_sources=7)
    S = wl.make_sources(w)
    zb = np.array([[32, 63, 0, 31, 64, 95], [5, 9, 70, 79, 0, 3]], dtype=np.int32)
    gen = {"seed": w.seed, "sources": S, "zero_boxes": zb, "continuum": w.continuum}
    a = H.Scene(w.dims, (32, 32, 32), gen=gen).host_cube()
    b = H.Scene(w.dims, (24, 16, 40), gen=gen).host_cube()
    assert np.array_equal(a, b)                     # bytes independent of the brick size
    from oracle import ovr
    ref = ovr.generate(w.seed, w.dims, sources=S, zero_boxes=zb, continuum=w.continuum)
    # both sides evaluate the same fp64 expression and round once to float32; the only freedom
    # left is the last bit of log / cos / exp in fp64, which can move a float32 rounding
    ulp = np.spacing(np.abs(ref).astype(np.float32))
    assert (np.abs(a - ref) <= ulp).all()
    assert np.mean(a == ref) > 0.9999
    assert (a[64:96, 0:32, 32:64] == 0).all() and (a[0:4, 70:80, 5:10] == 0).all()


# ------------------------------------------------------------------------------ closed forms on the GPU
def test_mip_axis_aligned_bit_exact(H):
    # BASELINE.json: "bit-exact for MIP under axis-aligned orthographic views"
    for dims, brick in [((64, 64, 64), (64, 64, 64)), ((40, 24, 56), (16, 16, 16)), ((33, 20, 17), (8, 12, 8))]:
        cube = noise_cube(dims[::-1], 3)
        cube[-1, -1, -1] = 40.0
        sc = H.Scene(dims, brick, cube=cube)
        vol = sc.oracle_volume()
        for axis in range(3):
            for sign in (1, -1):
                M, (W, Hh) = wl.axis_ortho_camera(dims, axis, sign)
                got = sc.render_mip(M, W, Hh, 0.5, miss=-1.0)
                ua, va = [(1, 2), (0, 2), (0, 1)][axis]
                assert np.array_equal(got[:dims[va], :dims[ua]], cube.max(axis=2 - axis))
                assert (got[dims[va]:] == -1.0).all() and (got[:, dims[ua]:] == -1.0).all()
                ref, _, _ = sc.ovr.render(vol, M, W, Hh, 0.5, sc.ovr.MIP, sc.ovr.F32, miss=-1.0)
                assert np.array_equal(got, ref)


def test_beer_lambert_and_ert_on_gpu(H):
    dims, step, a = (16, 16, 64), 0.5, 0.15
    rgb = np.array([0.2, 0.7, 0.5], dtype=np.float32)
    sc = H.Scene(dims, (16, 16, 16), cube=np.full(dims[::-1], 0.5, dtype=np.float32))
    t = np.zeros((256, 4), dtype=np.float32); t[:, :3] = rgb; t[:, 3] = a
    tf = (t, 0.0, 1.0)
    M, (W, Hh) = wl.axis_ortho_camera(dims, 2, 1)
    n = math.floor((dims[2] - 1) / step) + 1
    ap = 1.0 - (1.0 - a) ** step
    out = sc.render_ea(M, W, Hh, step, tf, tau=2.0)
    A = 1.0 - (1.0 - ap) ** n
    assert np.allclose(out[..., 3], A, atol=1e-5) and np.allclose(out[..., :3], rgb * A, atol=1e-5)
    sc.ctx.reset_counters()
    out = sc.render_ea(M, W, Hh, step, tf, tau=0.9)
    nstar = math.ceil(math.log(1.0 - 0.9) / math.log(1.0 - ap))
    c = sc.ctx.get_counters()
    assert c["taken_samples"] == nstar * W * Hh and c["rays_terminated"] == W * Hh
    assert c["nominal_samples"] == n * W * Hh
    assert (out[..., 3] >= 0.9).all() and (out[..., 3] <= 0.9 + 0.1 * ap + 1e-6).all()


def test_empty_cube_renders_background_bit_exact(H):
    dims = (40, 40, 40)
    sc = H.Scene(dims, (16, 16, 16), cube=np.zeros(dims[::-1], dtype=np.float32))
    M = wl.perspective_camera(dims, (70, 50))
    out = sc.render_ea(M, 70, 50, 0.5, wl.tf_src(), bg=BG, tau=0.99)
    assert np.array_equal(out, np.broadcast_to(np.array(BG, dtype=np.float32), out.shape))
    mip = sc.render_mip(M, 70, 50, 0.5, miss=-7.0)
    assert set(np.unique(mip)) == {0.0, -7.0}


# ------------------------------------------------------------------------------ BASELINE.json configs[0] (C1)
def test_config_c1_parity(H):
    w = wl.C1
    sc = H.Scene(w.dims, w.brick, gen={"seed": w.seed, "sources": wl.make_sources(w)})
    vol, ovr = sc.oracle_volume(), sc.ovr
    tf = wl.tf_ramp()
    W, Hh = w.frame
    for view in range(3):
        M = wl.config_camera(w, view)
        got = sc.render_ea(M, W, Hh, w.step, tf, bg=BG, tau=w.tau)
        o64, fl, _ = ovr.render(vol, M, W, Hh, w.step, ovr.EA, ovr.F64, tf=tf, bg=BG, tau=w.tau)
        o32, _, _ = ovr.render(vol, M, W, Hh, w.step, ovr.EA, ovr.F32, tf=tf, bg=BG, tau=w.tau)
        H.compare(got, o64, fl, o32, what=f"C1 EA view {view}")
        assert bit_fraction(got, o32) == 1.0
        mip, rgba = sc.render_mip(M, W, Hh, w.step, miss=0.0, tf=tf)
        m64, fl, _ = ovr.render(vol, M, W, Hh, w.step, ovr.MIP, ovr.F64, miss=0.0)
        m32, _, _ = ovr.render(vol, M, W, Hh, w.step, ovr.MIP, ovr.F32, miss=0.0)
        H.compare(mip, m64, fl, m32, mode_mip=True, vmin=tf[1], vmax=tf[2], miss=0.0, what=f"C1 MIP view {view}")
        assert bit_fraction(mip, m32) == 1.0
        # MIP colour = raw transfer function at the maximum
        j, i = np.unravel_index(np.argmax(mip), mip.shape)
        assert np.allclose(rgba[j, i], ovr.tf_lookup(tf, w.step, float(mip[j, i]), baked=False), atol=1e-6)
        assert (rgba[mip == 0.0] == 0).all() or (m64 != 0.0).all()


# ------------------------------------------------------------------------------ bricked, perspective (C2-like)
CASES = [
    ("c2-like", (96, 80, 128), (32, 32, 32), (160, 90), 0.5),
    ("ragged", (70, 45, 83), (24, 20, 32), (97, 61), 0.5),
    ("fine-step", (48, 48, 64), (16, 16, 16), (80, 64), 0.25),
    ("odd-step", (48, 40, 56), (16, 16, 16), (64, 48), 0.3),
]


@pytest.mark.parametrize("name,dims,brick,frame,step", CASES)
def test_bricked_perspective_parity(H, name, dims, brick, frame, step):
    w = wl.scaled(wl.C2, name, dims, brick, frame, n_sources=8)
    sc = H.Scene(dims, brick, gen={"seed": w.seed, "sources": wl.make_sources(w)})
    vol, ovr = sc.oracle_volume(), sc.ovr
    W, Hh = frame
    for az in (30.0, 200.0):
        M = wl.perspective_camera(dims, frame, azimuth_deg=az)
        for tfname, tau in (("src", 0.99), ("fog", 0.99), ("fog", 2.0)):
            tf = wl.TFS[tfname]()
            got = sc.render_ea(M, W, Hh, step, tf, bg=BG, tau=tau)
            o64, fl, c64 = ovr.render(vol, M, W, Hh, step, ovr.EA, ovr.F64, tf=tf, bg=BG, tau=tau)
            o32, _, _ = ovr.render(vol, M, W, Hh, step, ovr.EA, ovr.F32, tf=tf, bg=BG, tau=tau)
            H.compare(got, o64, fl, o32, what=f"{name} EA {tfname} tau={tau} az={az}")
            assert bit_fraction(got, o32) == 1.0, f"{name} EA {tfname}: not bit-identical to the float32 oracle"
        sc.ctx.reset_counters()
        mip = sc.render_mip(M, W, Hh, step, miss=-3.0)
        c = sc.ctx.get_counters()
        m64, fl, c64 = ovr.render(vol, M, W, Hh, step, ovr.MIP, ovr.F64, miss=-3.0)
        m32, _, c32 = ovr.render(vol, M, W, Hh, step, ovr.MIP, ovr.F32, miss=-3.0)
        H.compare(mip, m64, fl, m32, mode_mip=True, vmin=0.0, vmax=32.0, miss=-3.0, what=f"{name} MIP az={az}")
        assert bit_fraction(mip, m32) == 1.0
        assert c["nominal_samples"] == c32["nominal"]        # integer lattice invariant (O-3)


# ------------------------------------------------------------------------------ degenerate and awkward cases
def _check_both_paths(H, sc, vol, M, W, Hh, step, tf, tau, what, partition):
    """Whole-frame (GLOBAL) and sort-last EA + MIP of one view against the oracle, bit for bit in float32."""
    ovr, vr = sc.ovr, sc.vr
    got = sc.render_ea(M, W, Hh, step, tf, bg=BG, tau=tau)
    o64, fl, _ = ovr.render(vol, M, W, Hh, step, ovr.EA, ovr.F64, tf=tf, bg=BG, tau=tau)
    o32, _, _ = ovr.render(vol, M, W, Hh, step, ovr.EA, ovr.F32, tf=tf, bg=BG, tau=tau)
    H.compare(got, o64, fl, o32, what=what + " EA")
    assert np.array_equal(got, o32), what + " EA: not bit-identical to the float32 oracle"
    fr, _, _ = sc.render_sortlast(M, W, Hh, step, vr.MODE_EA, tf=tf, bg=BG, tau=tau)
    s32, _, _ = ovr.render(vol, M, W, Hh, step, ovr.EA, ovr.F32, tf=tf, bg=BG, tau=tau, split=ovr.SPLIT_SORTLAST, partition=partition)
    assert np.array_equal(fr, s32), what + " EA sort-last: not bit-identical to the float32 oracle"
    mip = sc.render_mip(M, W, Hh, step, miss=-1.0)
    m32, _, _ = ovr.render(vol, M, W, Hh, step, ovr.MIP, ovr.F32, miss=-1.0)
    assert np.array_equal(mip, m32), what + " MIP"
    mip_sl, _, _ = sc.render_sortlast(M, W, Hh, step, vr.MODE_MIP, bg=(-1.0, 0, 0, 0))
    assert np.array_equal(mip_sl, m32), what + " MIP sort-last"
    return got, mip


AWKWARD = [
    ("flat cube, one voxel thick", (40, 33, 1), (16, 16, 16), (64, 48), 0.5),
    ("two planes thick", (40, 33, 2), (16, 16, 16), (64, 48), 0.25),
    ("a single row of voxels", (57, 1, 1), (16, 8, 8), (48, 32), 0.25),
    ("bricks larger than the cube", (20, 24, 28), (64, 64, 64), (40, 40), 0.5),
    ("non-cubic bricks, ragged grid", (50, 37, 61), (32, 8, 16), (53, 41), 0.5),
    ("step longer than a voxel", (48, 48, 48), (16, 16, 16), (40, 40), 1.7),
    ("one-pixel frame", (32, 32, 32), (16, 16, 16), (1, 1), 0.5),
]


@pytest.mark.parametrize("name,dims,brick,frame,step", AWKWARD)
def test_awkward_shapes(H, name, dims, brick, frame, step):
    cube = noise_cube(dims[::-1], seed=11, scale=6.0) + 4.0
    sc = H.Scene(dims, brick, cube=cube)
    vol = sc.oracle_volume()
    W, Hh = frame
    part = tuple(min(b, n) for b, n in zip(brick, dims))
    for az, tf, tau in ((40.0, wl.tf_fog(), 0.99), (250.0, wl.tf_src(), 0.5)):
        M = wl.perspective_camera(dims, frame, azimuth_deg=az) if min(dims) > 1 else wl.perspective_camera(
            tuple(max(n, 2) for n in dims), frame, azimuth_deg=az)
        _check_both_paths(H, sc, vol, M, W, Hh, step, tf, tau, f"{name} az={az}", part)


def test_camera_inside_the_cube_and_rays_that_miss(H):
    dims, brick, frame = (64, 64, 64), (16, 16, 16), (72, 54)
    cube = noise_cube(dims[::-1], seed=3, scale=5.0) + 3.0
    sc = H.Scene(dims, brick, cube=cube)
    vol = sc.oracle_volume()
    W, Hh = frame
    # eye inside the cube: the near plane cuts the volume, rays start between voxels
    eye = np.array([30.3, 28.7, 17.2])
    V = wl._look_at(eye, eye + np.array([0.3, -0.2, 1.0]), np.array([0.0, 1.0, 0.0]))
    top = 0.75 * math.tan(math.radians(25.0))
    M = (wl._frustum(-top * W / Hh, top * W / Hh, -top, top, 0.75, 300.0) @ V).astype(np.float32)
    _check_both_paths(H, sc, vol, M, W, Hh, 0.5, wl.tf_fog(), 0.99, "eye inside", brick)
    # looking away from the cube: every ray misses, EA = background, MIP = miss value, bit for bit
    eye = np.array([32.0, 32.0, -80.0])
    V = wl._look_at(eye, eye + np.array([0.0, 0.0, -1.0]), np.array([0.0, 1.0, 0.0]))
    M = (wl._frustum(-top * W / Hh, top * W / Hh, -top, top, 0.75, 300.0) @ V).astype(np.float32)
    ea, mip = _check_both_paths(H, sc, vol, M, W, Hh, 0.5, wl.tf_fog(), 0.99, "all rays miss", brick)
    assert (ea == np.array(BG, np.float32)).all() and (mip == -1.0).all()


def test_extreme_transfer_functions(H):
    dims, brick, frame = (48, 40, 56), (16, 16, 16), (60, 44)
    cube = noise_cube(dims[::-1], seed=8, scale=4.0) + 10.0
    sc = H.Scene(dims, brick, cube=cube)
    vol = sc.oracle_volume()
    W, Hh = frame
    M = wl.perspective_camera(dims, frame, azimuth_deg=120.0)
    ramp = wl.tf_ramp()[0]
    clear = ramp.copy(); clear[:, 3] = 0.0                  # nothing is visible: the frame is the background
    ea, _ = _check_both_paths(H, sc, vol, M, W, Hh, 0.5, (clear, 0.0, 20.0), 0.99, "transparent table", brick)
    assert (ea == np.array(BG, np.float32)).all()
    solid = ramp.copy(); solid[:, 3] = 1.0                  # opaque at the first sample: alpha = 1 wherever the cube is hit
    ea, mip = _check_both_paths(H, sc, vol, M, W, Hh, 0.5, (solid, 0.0, 20.0), 0.99, "opaque table", brick)
    assert (ea[mip != -1.0][:, 3] == 1.0).all()
    _check_both_paths(H, sc, vol, M, W, Hh, 0.5, (ramp, 9.0, 9.5), 0.05, "narrow window, tau 0.05", brick)   # nearly everything clamps


def test_skipping_never_changes_a_frame(H):
    dims, brick, frame = (96, 96, 96), (16, 16, 16), (120, 90)
    w = wl.scaled(wl.C2, "skip", dims, brick, frame, n_sources=4)
    sc = H.Scene(dims, brick, gen={"seed": w.seed, "sources": wl.make_sources(w)})
    M = wl.perspective_camera(dims, frame)
    tf = wl.tf_src()
    res = {}
    for skip in (1, 0):
        sc.ctx.set_option(sc.vr.OPT_SKIP, skip)
        sc.ctx.reset_counters()
        ea = sc.render_ea(M, *frame, 0.5, tf, bg=BG, tau=0.99)
        c_ea = sc.ctx.get_counters()
        sc.ctx.reset_counters()
        mip = sc.render_mip(M, *frame, 0.5)
        c_mip = sc.ctx.get_counters()
        fr, _, ids = sc.render_sortlast(M, *frame, 0.5, sc.vr.MODE_EA, tf=tf, bg=BG, tau=2.0)
        res[skip] = (ea, mip, c_ea, c_mip, fr, len(ids))
    assert np.array_equal(res[0][0], res[1][0]) and np.array_equal(res[0][1], res[1][1])
    assert np.array_equal(res[0][4], res[1][4])
    assert res[1][2]["bricks_skipped"] > 0 and res[0][2]["bricks_skipped"] == 0
    assert res[1][2]["taken_samples"] < res[0][2]["taken_samples"]
    assert res[1][3]["taken_samples"] < res[0][3]["taken_samples"]
    assert res[1][5] < res[0][5]                       # inactive bricks drop out of the sort-last list
    assert res[1][2]["nominal_samples"] == res[0][2]["nominal_samples"]


# ------------------------------------------------------------------------------ S5 sort-last
@pytest.mark.parametrize("persp", [True, False])
def test_sort_last_partials_and_composite(H, persp):
    dims, brick, frame, step = (64, 48, 80), (32, 16, 32), (100, 70), 0.5
    cube = np.abs(noise_cube(dims[::-1], 5)) * 3.0
    sc = H.Scene(dims, brick, cube=cube)
    vol, ovr, vr = sc.oracle_volume(), sc.ovr, sc.vr
    tf = wl.tf_fog()
    M = wl.perspective_camera(dims, frame, azimuth_deg=130.0) if persp else \
        wl.ortho_camera(dims, frame, wl.seeded_directions(3, 1)[0])
    W, Hh = frame
    g = sc.grid()
    for mode, omode in ((vr.MODE_EA, ovr.EA), (vr.MODE_MIP, ovr.MIP)):
        for tau in ((0.9, 2.0) if mode == vr.MODE_EA else (2.0,)):
            fr, imgs, ids = sc.render_sortlast(M, W, Hh, step, mode, tf=tf, bg=BG, tau=tau)
            # visibility order: oracle keys non-decreasing along the library's order (O-9)
            keys, _ = ovr.visibility_keys(M, W, Hh, step, brick, g)
            assert (np.diff(keys[ids]) >= 0).all() and len(set(ids)) == len(ids)
            # a few partial images, bit for bit against the float32 oracle
            for q in (0, len(imgs) // 2, len(imgs) - 1):
                p = imgs[q]
                ref = ovr.render_brick(vol, M, W, Hh, step, omode, p["brick"], p["rect"], brick, ovr.F32, tf=tf, tau=tau)
                assert np.array_equal(p["image"], ref), (mode, tau, p["brick"])
            # every pixel outside a brick's rectangle must get nothing from that brick
            for p in imgs[:3]:
                full = ovr.render_brick(vol, M, W, Hh, step, omode, p["brick"], (0, 0, W, Hh), brick, ovr.F32, tf=tf, tau=tau)
                x0, y0, ww, hh = p["rect"]
                mask = np.ones((Hh, W), bool); mask[y0:y0 + hh, x0:x0 + ww] = False
                empty = (full[mask] == 0).all() if mode == vr.MODE_EA else np.isneginf(full[mask]).all()
                assert empty
            # the composited frame against the oracle's sort-last render (same mode, partition, tau)
            o32, _, _ = ovr.render(vol, M, W, Hh, step, omode, ovr.F32, tf=tf, bg=BG, tau=tau, miss=BG[0],
                                   split=ovr.SPLIT_SORTLAST, partition=brick)
            o64, fl, _ = ovr.render(vol, M, W, Hh, step, omode, ovr.F64, tf=tf, bg=BG, tau=tau, miss=BG[0],
                                    split=ovr.SPLIT_SORTLAST, partition=brick)
            assert np.array_equal(fr, o32)
            if mode == vr.MODE_EA:
                H.compare(fr, o64, fl, o32, what=f"sort-last EA tau={tau}")
            # split == unsplit (north_star closed form): MIP bit-exact, EA (ERT off) to 1e-6
            if mode == vr.MODE_MIP:
                assert np.array_equal(fr, sc.render_mip(M, W, Hh, step, miss=BG[0]))
            elif tau > 1.0:
                assert np.abs(fr - sc.render_ea(M, W, Hh, step, tf, bg=BG, tau=2.0)).max() < 1e-6
    # negative test: reversing the order of a near-opaque scene changes the frame
    fr_fwd, _, ids = sc.render_sortlast(M, W, Hh, step, vr.MODE_EA, tf=tf, bg=BG, tau=2.0)
    fr_rev, _, _ = sc.render_sortlast(M, W, Hh, step, vr.MODE_EA, tf=tf, bg=BG, tau=2.0, order=ids[::-1])
    assert np.abs(fr_fwd - fr_rev).max() > 1e-3


# ------------------------------------------------------------------------------ S6 tiled frame
def test_tiled_panels_into_one_pitched_frame(H):
    import torch
    dims, brick = (64, 64, 96), (32, 32, 32)
    w = wl.scaled(wl.C4, "tiles", dims, brick, (160, 90), n_sources=5)
    sc = H.Scene(dims, brick, gen={"seed": w.seed, "sources": wl.make_sources(w)})
    tf = wl.tf_fog()
    cols, rows, pw, ph = 5, 5, 32, 18
    W, Hh = cols * pw, rows * ph
    M = wl.perspective_camera(dims, (W, Hh))
    single = sc.render_ea(M, W, Hh, 0.25, tf, bg=BG, tau=0.99)
    frame = torch.full((Hh, W, 4), -7.0, dtype=torch.float32, device="cuda")
    sc.ctx.set_transfer_function(*tf)
    for r in range(rows):
        for c in range(cols):
            Mp = wl.panel_matrix(M, cols, rows, c, r)
            sc.ctx.set_view(Mp, pw, ph, 0.25)
            sc.ctx.set_viewport(c * pw, r * ph, W)
            sc.ctx.render_ea(frame, BG, 0.99)
    torch.cuda.synchronize()
    tiled = frame.cpu().numpy()
    assert (tiled != -7.0).all()
    assert np.abs(tiled - single).max() < 1e-4
    # one panel against the oracle with that panel's own matrix
    Mp = wl.panel_matrix(M, cols, rows, 2, 2)
    o32, _, _ = sc.ovr.render(sc.oracle_volume(), Mp, pw, ph, 0.25, sc.ovr.EA, sc.ovr.F32, tf=tf, bg=BG, tau=0.99)
    assert np.array_equal(tiled[2 * ph:3 * ph, 2 * pw:3 * pw], o32)


# ------------------------------------------------------------------------------ errors
def test_error_codes(H):
    import torch
    from paper_1012_2909_b200 import vr
    ctx = vr.Context(0)
    out = torch.zeros(16, 16, 4, device="cuda")
    with pytest.raises(vr.VRError) as e:
        ctx.render_ea(out)
    assert e.value.status == vr.ERR_STATE
    with pytest.raises(vr.VRError) as e:
        ctx.set_view(np.zeros(16, dtype=np.float32), 16, 16, 0.5)      # singular
    assert e.value.status == vr.ERR_INVALID_ARG
    with pytest.raises(vr.VRError) as e:
        ctx.set_view(np.eye(4, dtype=np.float32), 16, 16, 0.0)         # step <= 0
    assert e.value.status == vr.ERR_INVALID_ARG
    with pytest.raises(vr.VRError) as e:
        ctx.set_transfer_function(np.zeros((256, 4), dtype=np.float32), 1.0, 1.0)   # vmax <= vmin
    assert e.value.status == vr.ERR_INVALID_ARG
    ctx.set_view(np.eye(4, dtype=np.float32), 16, 16, 0.5)
    with pytest.raises(vr.VRError) as e:
        ctx.render_mip(out)                                            # still no cube
    assert e.value.status == vr.ERR_STATE


# ------------------------------------------------------------------------------ BASELINE.json full sizes
def _central_ray_axis(M):
    """Dominant axis of the ray through the frame centre (what VR_OPT_RING's default looks at)."""
    Mi = np.linalg.inv(np.asarray(M, dtype=np.float64).reshape(4, 4))
    pn, pf = Mi @ np.array([0, 0, -1.0, 1.0]), Mi @ np.array([0, 0, 1.0, 1.0])
    d = np.abs(pf[:3] / pf[3] - pn[:3] / pn[3])
    return int(np.argmax(d))


def _fullsize_check(H, w, block, n_random, frame_index, anchors=0, per_anchor=0):
    """Parity at a config's full size, in the launch configuration bench.py times (sort-last EA,
    plus whole-frame MIP): sampled pixels against the oracle (cube bytes fetched back brick by
    brick), and whole-frame properties that hold at any size.  `frame_index` may be a list of orbit
    frames (one resident cube).  Sampled pixels: a block at the frame centre, `n_random` seeded
    pixels that hit the cube anywhere in the frame, and `anchors` seeded hit pixels spread over the
    whole frame with `per_anchor` pixels drawn from the 9 x 9 neighbourhood of each (neighbouring
    rays cross the same bricks, so a 64 GiB cube is checked far from the frame centre for a few GB of
    traffic; the bricks of one anchor are dropped before the next is fetched)."""
    import torch
    from oracle import ovr
    sc = H.Scene(w.dims, w.brick, gen={"seed": w.seed, "sources": wl.make_sources(w),
                                       "zero_boxes": wl.make_zero_boxes(w), "continuum": w.continuum})
    vr = sc.vr
    W, Hh = w.frame
    tf = wl.TFS[w.tf]()
    brick = tuple(min(b, n) for b, n in zip(w.brick, w.dims))
    rng = np.random.default_rng(w.view_seed)
    frames = list(frame_index) if isinstance(frame_index, (list, tuple)) else [frame_index]
    axes = []
    for fi in frames:
        M = wl.config_camera(w, fi)
        axes.append(_central_ray_axis(M))
        frame, imgs, ids = sc.render_sortlast(M, W, Hh, w.step, vr.MODE_EA, tf=tf, bg=BG, tau=w.tau)
        mip = sc.render_mip(M, W, Hh, w.step, miss=0.0)
        cx, cy = W // 2, Hh // 2
        xs, ys = np.arange(cx - block // 2, cx + block // 2), np.arange(cy - block // 2, cy + block // 2)
        groups = [np.stack(np.meshgrid(xs, ys), axis=-1).reshape(-1, 2)]
        hit = np.argwhere(mip != 0.0)
        if n_random:
            pick = hit[rng.choice(len(hit), size=min(n_random, len(hit)), replace=False)]
            groups[0] = np.concatenate([groups[0], pick[:, ::-1]])
        for a in hit[rng.choice(len(hit), size=min(anchors, len(hit)), replace=False)] if anchors else []:
            dx, dy = rng.integers(-4, 5, size=per_anchor), rng.integers(-4, 5, size=per_anchor)
            px = np.stack([np.clip(a[1] + dx, 0, W - 1), np.clip(a[0] + dy, 0, Hh - 1)], axis=-1)
            groups.append(np.unique(px, axis=0))
        n_checked, off_centre_bricks = 0, set()
        pool = {"ea": [], "mip": []}
        for pix in groups:
            pix = pix.astype(np.int32)
            touched = ovr.bricks_touched(M, W, Hh, w.step, w.dims, brick, pix)
            off_centre_bricks.update(int(b) for b in touched)
            vol = ovr.Volume(w.dims, brick, {int(b): sc.download_brick(int(b)) for b in touched})
            kw = dict(tf=tf, bg=BG, tau=w.tau, pixels=pix)
            o64, fl, _ = ovr.render(vol, M, W, Hh, w.step, ovr.EA, ovr.F64, split=ovr.SPLIT_SORTLAST, partition=brick, **kw)
            o32, _, _ = ovr.render(vol, M, W, Hh, w.step, ovr.EA, ovr.F32, split=ovr.SPLIT_SORTLAST, partition=brick, **kw)
            got = frame[pix[:, 1], pix[:, 0]]
            assert np.array_equal(got, o32)                   # the kernels implement the float32 reading to the bit
            pool["ea"].append((got, o64, fl, o32))
            m64, flm, _ = ovr.render(vol, M, W, Hh, w.step, ovr.MIP, ovr.F64, miss=0.0, pixels=pix)
            m32, _, _ = ovr.render(vol, M, W, Hh, w.step, ovr.MIP, ovr.F32, miss=0.0, pixels=pix)
            gm = mip[pix[:, 1], pix[:, 0]]
            assert np.array_equal(gm, m32)
            pool["mip"].append((gm, m64, flm, m32))
            n_checked += len(pix)
            del vol
        # BASELINE.json's tolerances are per frame and channel: all sampled pixels of the frame pooled
        ea, mp = ([np.concatenate(v) for v in zip(*pool[k])] for k in ("ea", "mip"))
        st_ea = H.compare(*ea, what=f"{w.name} full-size EA sort-last, frame {fi}")
        st_mip = H.compare(*mp, mode_mip=True, vmin=tf[1], vmax=tf[2], miss=0.0, what=f"{w.name} full-size MIP, frame {fi}")
        print(f"[parity] {w.name} frame {fi}: {n_checked} pixels, {len(off_centre_bricks)} bricks; EA max {st_ea['max'].max():.2e} rms "
              f"{st_ea['rms'].max():.2e}; MIP max {st_mip['max'].max():.2e} rms {st_mip['rms'].max():.2e} (of 1e-4 / 1e-5)")
        assert n_checked >= block * block + n_random + anchors * max(1, per_anchor // 3)
        # whole-frame properties: MIP split == unsplit bit-exact (so the sort-last MIP frame equals the oracle on the
        # sampled pixels too); EA sort-last (ERT off) == global to 1e-6;
        # ERT bound |frame_tau - frame_inf| <= (1 - tau) / tau; alpha within [0, 1]
        mip_sl, _, _ = sc.render_sortlast(M, W, Hh, w.step, vr.MODE_MIP, bg=(0.0, 0, 0, 0))
        assert np.array_equal(mip_sl, mip)
        sl_inf, _, _ = sc.render_sortlast(M, W, Hh, w.step, vr.MODE_EA, tf=tf, bg=BG, tau=2.0)
        gl_inf = sc.render_ea(M, W, Hh, w.step, tf, bg=BG, tau=2.0)
        assert np.abs(sl_inf - gl_inf).max() < 2e-6
        assert np.abs(frame - sl_inf).max() <= (1 - w.tau) / w.tau + 1e-6
        assert frame[..., 3].min() >= 0.0 and frame[..., 3].max() <= 1.0 + 1e-6
        if anchors:        # the anchors reach bricks whose byte offset in the brick-major cube passes 2^32
            vox = brick[0] * brick[1] * brick[2]
            assert max(off_centre_bricks) * vox * 4 > 2 ** 32 or w.n_voxels * 4 <= 2 ** 32
    del sc
    torch.cuda.empty_cache()
    return axes


def test_config_c2_full_size(H, marcher):
    if marcher not in ("auto", "v0"):
        pytest.skip("full sizes run with the library's choice (what bench.py times) and variant 0")
    _fullsize_check(H, wl.C2, block=16, n_random=200, frame_index=0)


def test_config_c3_full_size_64gib(H, marcher):
    if marcher not in ("auto", "v0", "v3t"):
        pytest.skip("full sizes run with the library's choice (what bench.py times), variant 0 and the object-order MIP")
    import torch
    torch.cuda.empty_cache()
    free, total = torch.cuda.mem_get_info()
    if free < 80e9:
        pytest.skip("needs ~70 GB of free HBM")
    # two orbit frames: the central ray runs mostly along z, the short axis of the micro-blocks, on one and along x on
    # the other (the two extremes of the gather pattern; the library's ring form, registers on this layout, serves both -
    # the cp.async form is compared with the oracle under the forced "v3s" / "v3d" plans); seeded hit pixels over the frame
    axes = _fullsize_check(H, wl.C3, block=12, n_random=0, frame_index=[0, 90], anchors=12, per_anchor=24)
    assert (axes[0] == 2) != (axes[1] == 2), axes


def test_hipass_shaped_cube_with_partial_edge_bricks(H, marcher):
    """PAPER.md line 57 (footnote 4): the HIPASS southern-sky cube is 1721 x 1721 x 1025 float32
    ("12 GB"); line 61: it is shown rendered at 3000 x 3000.  The real cube is not in the
    container: a synthetic cube of that shape (the C3 recipe, 3000 sources), whose dimensions are
    no multiple of the 256^3 bricks, so every face of the brick grid has partial bricks."""
    if marcher != "auto":
        pytest.skip("run once, with the library's choice")
    import torch
    torch.cuda.empty_cache()
    free, total = torch.cuda.mem_get_info()
    if free < 20e9:
        pytest.skip("needs ~14 GB of free HBM")
    w = wl.scaled(wl.C3, "HIPASS-shaped", (1721, 1721, 1025), (256, 256, 256), (3000, 3000), n_sources=3000)
    assert w.brick_grid == (7, 7, 5)
    _fullsize_check(H, w, block=10, n_random=80, frame_index=25)


def _tiled_fullsize_check(H, w, panels, block, mip_frame=None):
    """Parity at the full size of a tiled-display config (BASELINE.json configs[3], configs[4];
    PAPER.md line 37: 5 x 5 panels of 1920 x 1080), in the launch configuration bench.py times:
    every panel is an off-axis frustum of the one camera, rendered sort-last into one pitched
    frame.  Pixel blocks of the listed panels are compared with the oracle run with the panel's
    matrix, the cube bytes fetched back brick by brick.  Optionally a whole-cube MIP at `mip_frame` (configs[4])."""
    import torch
    from oracle import ovr
    sc = H.Scene(w.dims, w.brick, gen={"seed": w.seed, "sources": wl.make_sources(w),
                                       "zero_boxes": wl.make_zero_boxes(w), "continuum": w.continuum})
    vr = sc.vr
    W, Hh = w.frame
    cols, rows = w.panels
    pw, ph = W // cols, Hh // rows
    M = wl.config_camera(w, 0)
    tf = wl.TFS[w.tf]()
    sc.ctx.set_transfer_function(*tf)
    frame = torch.full((Hh, W, 4), -7.0, dtype=torch.float32, device="cuda")
    arena = None
    n_bricks = 0
    for r in range(rows):
        for c in range(cols):
            sc.ctx.set_view(wl.panel_matrix(M, cols, rows, c, r), pw, ph, w.step)
            sc.ctx.set_viewport(c * pw, r * ph, W)
            ids = sc.ctx.sort_bricks(vr.MODE_EA)
            parts, n, nbytes = sc.ctx.partial_layout(vr.MODE_EA, ids)
            if arena is None or arena.numel() < nbytes:
                arena = torch.empty(int(nbytes * 1.3) + 256, dtype=torch.uint8, device="cuda")
            vr.Context.bind_partials(parts, n, arena)
            sc.ctx.render_bricks(vr.MODE_EA, parts, n, w.tau)
            sc.ctx.composite_bricks(vr.MODE_EA, parts, n, frame, BG)
            n_bricks += n
    torch.cuda.synchronize()
    assert n_bricks > 0
    brick = tuple(min(b, n) for b, n in zip(w.brick, w.dims))
    cache = {}
    rng = np.random.default_rng(w.view_seed)
    n_checked = 0
    for (c, r) in panels:
        # the block in the panel's lower right corner (next to the seams), cast by the oracle with
        # the panel's own off-axis matrix: same rays, so the float32 oracle must match to the bit
        Mp = wl.panel_matrix(M, cols, rows, c, r)
        bx, by = int(rng.integers(0, pw - block + 1)), int(rng.integers(0, ph - block + 1))
        for (ox, oy) in ((pw - block, ph - block), (bx, by)):          # ... and a block at a seeded place inside the panel
            xs, ys = np.arange(ox, ox + block), np.arange(oy, oy + block)
            pix = np.stack(np.meshgrid(xs, ys), axis=-1).reshape(-1, 2).astype(np.int32)
            touched = ovr.bricks_touched(Mp, pw, ph, w.step, w.dims, brick, pix)
            if len(cache) + len(touched) > 48:
                cache.clear()                                           # bound the host copy of the cube
            for b in touched:
                if int(b) not in cache:
                    cache[int(b)] = sc.download_brick(int(b))
            vol = ovr.Volume(w.dims, brick, {int(b): cache[int(b)] for b in touched})
            kw = dict(tf=tf, bg=BG, tau=w.tau, pixels=pix, split=ovr.SPLIT_SORTLAST, partition=brick)
            o64, fl, _ = ovr.render(vol, Mp, pw, ph, w.step, ovr.EA, ovr.F64, **kw)
            o32, _, _ = ovr.render(vol, Mp, pw, ph, w.step, ovr.EA, ovr.F32, **kw)
            got = frame[r * ph + ys[0]:r * ph + ys[-1] + 1, c * pw + xs[0]:c * pw + xs[-1] + 1].cpu().numpy().reshape(-1, 4)
            H.compare(got, o64, fl, o32, what=f"{w.name} full-size tiled EA, panel {(c, r)} block at {(ox, oy)}")
            assert np.array_equal(got, o32)
            n_checked += len(pix)
    # whole-frame properties: every pixel written, alpha in [0, 1], rows continuous across panel seams
    lo, hi = torch.aminmax(frame[..., 3])
    assert float(lo) >= min(0.0, BG[3]) and float(hi) <= 1.0 + 1e-6
    assert not bool((frame == -7.0).any())
    for r in range(1, rows):
        seam = (frame[r * ph] - frame[r * ph - 1]).abs().mean()
        inner = (frame[r * ph + 1] - frame[r * ph]).abs().mean()
        assert float(seam) < 4.0 * float(inner) + 1e-3
    if mip_frame is not None:
        mw, mh = mip_frame
        Mm = wl.config_camera(w, 0, frame=mip_frame)
        mip = sc.render_mip(Mm, mw, mh, w.step, miss=0.0)
        mip_sl, _, _ = sc.render_sortlast(Mm, mw, mh, w.step, vr.MODE_MIP, bg=(0.0, 0, 0, 0))
        assert np.array_equal(mip_sl, mip)                      # split == unsplit, bit-exact (O-5)
        xs, ys = np.arange(mw // 2 - 12, mw // 2 + 12), np.arange(mh // 2 - 12, mh // 2 + 12)
        pix = np.stack(np.meshgrid(xs, ys), axis=-1).reshape(-1, 2).astype(np.int32)
        touched = ovr.bricks_touched(Mm, mw, mh, w.step, w.dims, brick, pix)
        for b in touched:
            if int(b) not in cache:
                cache[int(b)] = sc.download_brick(int(b))
        vol = ovr.Volume(w.dims, brick, {int(b): cache[int(b)] for b in touched})
        m64, flm, _ = ovr.render(vol, Mm, mw, mh, w.step, ovr.MIP, ovr.F64, miss=0.0, pixels=pix)
        m32, _, _ = ovr.render(vol, Mm, mw, mh, w.step, ovr.MIP, ovr.F32, miss=0.0, pixels=pix)
        gm = mip[pix[:, 1], pix[:, 0]]
        H.compare(gm, m64, flm, m32, mode_mip=True, vmin=tf[1], vmax=tf[2], miss=0.0, what=f"{w.name} full-size MIP")
        assert np.array_equal(gm, m32)
    del sc, frame, arena
    torch.cuda.empty_cache()


def test_config_c4_full_size_tiled_9600x5400(H, marcher):
    if marcher != "auto":
        pytest.skip("full sizes run with the library's choice (what bench.py times)")
    _tiled_fullsize_check(H, wl.C4, panels=[(2, 2), (0, 1), (4, 3), (2, 0)], block=8)


def test_config_c5_full_size_128gib(H, marcher):
    if marcher != "auto":
        pytest.skip("full sizes run with the library's choice (what bench.py times)")
    import torch
    torch.cuda.empty_cache()
    free, total = torch.cuda.mem_get_info()
    if free < 150e9:
        pytest.skip("needs ~142 GB of free HBM")
    _tiled_fullsize_check(H, wl.C5, panels=[(2, 2), (1, 3), (3, 1)], block=6, mip_frame=(1920, 1080))


def test_upload_refuses_non_finite_voxels(H):
    import torch
    from paper_1012_2909_b200 import vr
    dims, brick = (20, 12, 9), (8, 8, 8)
    for bad in (np.nan, np.inf, -np.inf):
        cube = noise_cube(dims[::-1], seed=2)
        cube[4, 7, 13] = bad
        cb, mb = vr.cube_layout(dims, brick)
        d_cube = torch.empty(cb // 4, dtype=torch.float32, device="cuda")
        d_meta = torch.empty(mb, dtype=torch.uint8, device="cuda")
        ctx = vr.Context(0)
        with pytest.raises(vr.VRError) as e:
            ctx.upload_cube(cube, dims, brick, d_cube, d_meta)
        assert e.value.status == vr.ERR_INVALID_ARG and "non-finite" in str(e.value)
        with pytest.raises(vr.VRError) as e:                      # and the same from device memory
            ctx.upload_cube(torch.from_numpy(cube).cuda(), dims, brick, d_cube, d_meta)
        assert e.value.status == vr.ERR_INVALID_ARG
        ctx.set_view(np.eye(4, dtype=np.float32), 8, 8, 0.5)
        out = torch.empty((8, 8), dtype=torch.float32, device="cuda")
        with pytest.raises(vr.VRError) as e:
            ctx.render_mip(out)                                     # no cube was set
        assert e.value.status == vr.ERR_STATE


def test_brick_and_macro_cell_minmax_against_numpy(H):
    """S0 metadata (white box: d_meta starts with (min,max) per brick, then per 8^3 macro-cell, each
    region 256-byte aligned): min / max over the region's voxels plus the +1 layer, clipped to the
    cube (O-10: halo-inclusive, so that a trilinear footprint is always covered)."""
    dims, brick = (45, 38, 29), (16, 24, 8)
    cube = noise_cube(dims[::-1], seed=21, scale=3.0)
    sc = H.Scene(dims, brick, cube=cube)
    sc.torch.cuda.synchronize()
    meta = sc.d_meta.cpu().numpy()
    g = sc.grid()
    nb = g[0] * g[1] * g[2]
    C = [-(-b // 8) for b in brick]
    cpb = C[0] * C[1] * C[2]
    bmm = meta[:8 * nb].view(np.float32).reshape(nb, 2)
    off = -(-8 * nb // 256) * 256
    cmm = meta[off:off + 8 * nb * cpb].view(np.float32).reshape(nb, cpb, 2)
    for bid in range(nb):
        bi = (bid % g[0], (bid // g[0]) % g[1], bid // (g[0] * g[1]))
        o = [bi[a] * brick[a] for a in range(3)]
        hi = [min(o[a] + brick[a], dims[a] - 1) for a in range(3)]               # inclusive, +1 layer, inside the cube
        reg = cube[o[2]:hi[2] + 1, o[1]:hi[1] + 1, o[0]:hi[0] + 1]
        assert bmm[bid, 0] == reg.min() and bmm[bid, 1] == reg.max(), bid
        for cz in range(C[2]):
            for cy in range(C[1]):
                for cx in range(C[0]):
                    lo = [o[0] + 8 * cx, o[1] + 8 * cy, o[2] + 8 * cz]
                    h2 = [min(lo[a] + 8, o[a] + brick[a], dims[a] - 1) for a in range(3)]
                    got = cmm[bid, cx + C[0] * (cy + C[1] * cz)]
                    if any(h2[a] < lo[a] for a in range(3)):
                        assert got[0] > got[1]                                    # empty cell: (inf, -inf)
                        continue
                    r = cube[lo[2]:h2[2] + 1, lo[1]:h2[1] + 1, lo[0]:h2[0] + 1]
                    assert got[0] == r.min() and got[1] == r.max(), (bid, cx, cy, cz)


def test_occupancy_bits_against_numpy(H, marcher):
    """S1 classification at the finest level (white box: d_meta holds (min,max) per brick and per macro-cell, the
    macro-cell bits, the brick flags, then one occupancy word per 128-byte line of the cube, each region 256-byte
    aligned): the bit of the trilinear cell with lower corner (lx, ly, lz), slot (lx&3) + 4 (ly&1) + 8 (lz&1) +
    16 ((ly>>1)&1) of micro-block (lx>>2, ly>>2, lz>>1), is set iff one of the cell's 8 corners (zeros beyond the
    cube) maps above the table's transparent prefix, (v - vmin) * scale > t in float32 (O-10)."""
    if marcher != "auto":
        pytest.skip("the classification does not depend on the marcher")
    dims, brick = (45, 38, 29), (16, 24, 8)
    cube = noise_cube(dims[::-1], seed=33, scale=2.0)
    sc = H.Scene(dims, brick, cube=cube)
    vr = sc.vr
    sc.ctx.set_option(vr.OPT_VARIANT, 0)
    tfs = wl.tf_src(24)
    M = wl.perspective_camera(dims, (64, 48), azimuth_deg=20.0)
    sc.render_ea(M, 64, 48, 0.5, tfs, tau=0.99)                    # classifies against the table
    assert sc.ctx.get_plan(vr.MODE_EA)["skip_level"] == 3
    meta = sc.d_meta.cpu().numpy()
    g = sc.grid()
    nb = g[0] * g[1] * g[2]
    C = [-(-b // 8) for b in brick]
    cpb = C[0] * C[1] * C[2]
    T = [(brick[0] + 4) // 4, (brick[1] + 4) // 4, (brick[2] + 2) // 2]
    per = T[0] * T[1] * T[2]
    up = lambda v: -(-v // 256) * 256
    off = up(8 * nb)
    off = up(off + 8 * nb * cpb)
    off = up(off + 4 * nb * ((cpb + 31) // 32))
    off = up(off + 4 * nb)
    occ = meta[off:off + 4 * nb * per].view(np.uint32).reshape(nb, per)
    pad = np.zeros((dims[2] + 1, dims[1] + 1, dims[0] + 1), dtype=np.float32)
    pad[:-1, :-1, :-1] = cube
    scale = np.float32(255.0 / (tfs[2] - tfs[1]))
    hot = ((pad - np.float32(tfs[1])) * scale) > np.float32(24.0)
    want = np.zeros_like(hot[:-1, :-1, :-1])
    for dz in (0, 1):
        for dy in (0, 1):
            for dx in (0, 1):
                want |= hot[dz:dz + dims[2], dy:dy + dims[1], dx:dx + dims[0]]
    n_set = 0
    for bid in range(nb):
        bi = (bid % g[0], (bid // g[0]) % g[1], bid // (g[0] * g[1]))
        o = [bi[a] * brick[a] for a in range(3)]
        ext = [min(brick[a], dims[a] - o[a]) for a in range(3)]
        lx, ly, lz = np.meshgrid(np.arange(ext[0]), np.arange(ext[1]), np.arange(ext[2]), indexing="ij")
        word = (lx >> 2) + T[0] * ((ly >> 2) + T[1] * (lz >> 1))
        bit = (lx & 3) + 4 * (ly & 1) + 8 * (lz & 1) + 16 * ((ly >> 1) & 1)
        got = (occ[bid][word] >> bit.astype(np.uint32)) & 1
        ref = want[o[2] + lz, o[1] + ly, o[0] + lx]
        assert np.array_equal(got.astype(bool), ref), bid
        n_set += int(ref.sum())
    assert 0 < n_set < want.size // 2


@pytest.mark.parametrize("mode_name", ["ea", "mip"])
def test_render_sortlast_one_call_equals_the_four_calls(H, marcher, mode_name):
    """vr_render_sortlast = vr_sort_bricks + vr_partial_layout + vr_render_bricks + vr_composite_bricks: same frame, bit
    for bit; an arena that is too small is refused with the size it needs and nothing is rendered."""
    import torch
    w = wl.scaled(wl.C2, "one", (96, 80, 112), (32, 32, 32), (160, 100), n_sources=10)
    sc = H.Scene(w.dims, w.brick, gen={"seed": w.seed, "sources": wl.make_sources(w)})
    vr = sc.vr
    mode = vr.MODE_EA if mode_name == "ea" else vr.MODE_MIP
    W, Hh = w.frame
    tf = wl.tf_src(20)
    bg = BG if mode == vr.MODE_EA else (-2.0, 0, 0, 0)
    for az in (15.0, 140.0):
        M = wl.perspective_camera(w.dims, w.frame, azimuth_deg=az)
        ref, _, ids = sc.render_sortlast(M, W, Hh, 0.5, mode, tf=tf, bg=bg, tau=0.9)
        ch = 4 if mode == vr.MODE_EA else 1
        out = torch.full((Hh, W, ch), -7.0, dtype=torch.float32, device="cuda")
        ok, need = sc.ctx.render_sortlast(mode, None, out, bg, 0.9)
        assert not ok and need > 0 and float(out.min()) == -7.0
        small = torch.empty(need - 256, dtype=torch.uint8, device="cuda")
        assert sc.ctx.render_sortlast(mode, small, out, bg, 0.9) == (False, need)
        arena = torch.empty(need, dtype=torch.uint8, device="cuda")
        assert sc.ctx.render_sortlast(mode, arena, out, bg, 0.9) == (True, need)
        torch.cuda.synchronize()
        got = out.cpu().numpy()
        assert np.array_equal(got if ch == 4 else got[..., 0], ref)
