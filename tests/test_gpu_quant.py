"""float16 cube storage on the GPU (VR_OPT_VOXEL_TYPE 1, O-16) against the oracle's
definition: the stored cube is oracle/oquant.quantise_f16 of the float32 cube, bit for bit, and every marcher renders
it exactly as the float32 oracle renders that dequantised cube.  The distance to the UNquantised frame is checked
against the bound O-16 derives (MIP) and the looser tolerance it states (emission-absorption)."""
import numpy as np
import pytest

from paper_1012_2909_b200 import workloads as wl

pytestmark = pytest.mark.gpu

BG = (0.25, 0.5, 0.125, 0.75)
QTOL_EA_MAX, QTOL_EA_RMS = 2e-3, 2e-4          # DESIGN.md O-16: float16 cube vs float32 cube, per channel in [0, 1]


@pytest.fixture(scope="module")
def H():
    import helpers
    helpers.torch_cuda()
    return helpers


@pytest.fixture(params=["auto", "v0", "v1", "v3s", "v3d", "v3o", "v4o"])
def plan(request, H):
    from paper_1012_2909_b200 import vr
    H.FORCED_OPTIONS.clear()
    H.FORCED_OPTIONS[vr.OPT_VOXEL_TYPE] = vr.VOXEL_F16
    if request.param != "auto":
        H.FORCED_OPTIONS.update({vr.OPT_VARIANT: int(request.param[1]), vr.OPT_CELL_SKIP: 1})
        if request.param[2:]:
            H.FORCED_OPTIONS[vr.OPT_DENSE] = int(request.param[2] == "d")
            H.FORCED_OPTIONS[vr.OPT_OCCUPANCY] = int(request.param[2] == "o")
    yield request.param
    H.FORCED_OPTIONS.clear()


def test_stored_cube_is_the_oracles_quantisation(H, plan):
    if plan != "auto":
        pytest.skip("storage does not depend on the marcher")
    from oracle import ovr, oquant
    # uploaded from a float32 array (host and device source), ragged bricks
    dims, brick = (37, 29, 41), (16, 16, 16)
    cube = (np.random.default_rng(1).normal(size=dims[::-1]) * 7.0).astype(np.float32)
    sc = H.Scene(dims, brick, cube=cube)
    assert np.array_equal(sc.host_cube(), oquant.quantise_f16(cube))
    # generated on the device: the float32 generator output, then the same rounding
    w = wl.scaled(wl.C3, "qgen", (96, 80, 64), (32, 32, 32), (64, 64), n_sources=9)
    S = wl.make_sources(w)
    sg = H.Scene(w.dims, w.brick, gen={"seed": w.seed, "sources": S, "continuum": w.continuum})
    ref = ovr.generate(w.seed, w.dims, sources=S, continuum=w.continuum)
    got = sg.host_cube()
    want = oquant.quantise_f16(ref)
    # the device evaluates log / cos / exp in fp64 with possibly different last bits: <= 1 ulp of float32 before the
    # rounding to float16, i.e. at most one float16 step apart, and equal almost everywhere
    assert np.mean(got == want) > 0.999
    assert (np.abs(got.astype(np.float64) - want) <= 2.0 ** -10 * np.abs(want) + 2.0 ** -24).all()
    # half the bytes
    cb32, _ = sc.vr.cube_layout_typed(w.dims, w.brick, sc.vr.VOXEL_F32)
    cb16, _ = sc.vr.cube_layout_typed(w.dims, w.brick, sc.vr.VOXEL_F16)
    assert cb16 * 2 == cb32


def test_out_of_range_voxels_are_refused(H, plan):
    if plan != "auto":
        pytest.skip("storage does not depend on the marcher")
    import torch
    from paper_1012_2909_b200 import vr
    dims, brick = (20, 12, 9), (8, 8, 8)
    cube = np.zeros(dims[::-1], np.float32)
    cube[4, 7, 13] = 1.0e5                                  # finite in float32, infinite in float16
    cb, mb = vr.cube_layout(dims, brick)
    ctx = vr.Context(0)
    ctx.set_option(vr.OPT_VOXEL_TYPE, vr.VOXEL_F16)
    with pytest.raises(vr.VRError) as e:
        ctx.upload_cube(cube, dims, brick, torch.empty(cb // 4, device="cuda"), torch.empty(mb, dtype=torch.uint8, device="cuda"))
    assert e.value.status == vr.ERR_INVALID_ARG
    with pytest.raises(vr.VRError):
        ctx.set_option(vr.OPT_LAYOUT, 0)                    # float16 needs the micro-block layout


@pytest.mark.parametrize("persp", [True, False])
def test_every_marcher_renders_the_dequantised_cube_like_the_oracle(H, plan, persp):
    from oracle import ovr, oquant
    w = wl.scaled(wl.C2, "q16", (80, 72, 96), (32, 32, 32), (120, 90), n_sources=10)
    S = wl.make_sources(w)
    sc = H.Scene(w.dims, w.brick, gen={"seed": w.seed, "sources": S})
    vr = sc.vr
    W, Hh = w.frame
    M = wl.perspective_camera(w.dims, w.frame, azimuth_deg=50.0) if persp else wl.ortho_camera(w.dims, w.frame, wl.seeded_directions(5, 1)[0])
    vol = sc.oracle_volume()                                   # the dequantised bytes as they sit on the device
    for tf, tau in ((wl.tf_src(20), 0.95), (wl.tf_fog(), 0.9)):
        ea = sc.render_ea(M, W, Hh, 0.5, tf, bg=BG, tau=tau)
        o32, _, _ = ovr.render(vol, M, W, Hh, 0.5, ovr.EA, ovr.F32, tf=tf, bg=BG, tau=tau)
        o64, fl, _ = ovr.render(vol, M, W, Hh, 0.5, ovr.EA, ovr.F64, tf=tf, bg=BG, tau=tau)
        assert np.array_equal(ea, o32), plan
        H.compare(ea, o64, fl, o32, what=f"float16 cube EA {plan}")
        fr, _, _ = sc.render_sortlast(M, W, Hh, 0.5, vr.MODE_EA, tf=tf, bg=BG, tau=tau)
        s32, _, _ = ovr.render(vol, M, W, Hh, 0.5, ovr.EA, ovr.F32, tf=tf, bg=BG, tau=tau, split=ovr.SPLIT_SORTLAST, partition=w.brick)
        assert np.array_equal(fr, s32), plan
    mip = sc.render_mip(M, W, Hh, 0.5, miss=-1.0)
    m32, _, _ = ovr.render(vol, M, W, Hh, 0.5, ovr.MIP, ovr.F32, miss=-1.0)
    assert np.array_equal(mip, m32), plan
    mip_sl, _, _ = sc.render_sortlast(M, W, Hh, 0.5, vr.MODE_MIP, bg=(-1.0, 0, 0, 0))
    assert np.array_equal(mip_sl, mip)
    # against the UNquantised cube (the oracle's float32 generator output): the O-16 bound for MIP, the stated
    # tolerance for emission-absorption
    ref_cube = ovr.generate(w.seed, w.dims, sources=S)
    rvol = ovr.Volume.linear(ref_cube)
    r_mip, _, _ = ovr.render(rvol, M, W, Hh, 0.5, ovr.MIP, ovr.F64, miss=-1.0)
    hit = r_mip != -1.0
    bound = 2.0 ** -11 * np.abs(ref_cube).max() + 2.0 ** -10 * np.abs(ref_cube).max() + 1e-5      # + the generator's last-bit freedom
    assert (np.abs(mip[hit].astype(np.float64) - r_mip[hit]) <= bound).all()
    tf = wl.tf_src(20)
    r_ea, _, _ = ovr.render(rvol, M, W, Hh, 0.5, ovr.EA, ovr.F64, tf=tf, bg=BG, tau=2.0)
    q_ea = sc.render_ea(M, W, Hh, 0.5, tf, bg=BG, tau=2.0)
    err = np.abs(q_ea.astype(np.float64) - r_ea)
    assert err.max() <= QTOL_EA_MAX and np.sqrt((err ** 2).mean(axis=(0, 1))).max() <= QTOL_EA_RMS
    assert err.max() > 0.0                                     # and it IS a different cube


def test_meta_and_occupancy_follow_the_dequantised_values(H, plan):
    if plan != "auto":
        pytest.skip("classification does not depend on the marcher")
    dims, brick = (45, 38, 29), (16, 24, 8)
    cube = (np.random.default_rng(21).normal(size=dims[::-1]) * 3.0).astype(np.float32)
    sc = H.Scene(dims, brick, cube=cube)
    q = sc.host_cube()
    meta = sc.d_meta.cpu().numpy()
    g = sc.grid()
    nb = g[0] * g[1] * g[2]
    bmm = meta[:8 * nb].view(np.float32).reshape(nb, 2)
    for bid in range(nb):
        bi = (bid % g[0], (bid // g[0]) % g[1], bid // (g[0] * g[1]))
        o = [bi[a] * brick[a] for a in range(3)]
        hi = [min(o[a] + brick[a], dims[a] - 1) for a in range(3)]
        reg = q[o[2]:hi[2] + 1, o[1]:hi[1] + 1, o[0]:hi[0] + 1]
        assert bmm[bid, 0] == reg.min() and bmm[bid, 1] == reg.max(), bid
    # skipping on / off give the same frame on the quantised cube too (the occupancy bits come from the same values)
    vr = sc.vr
    M = wl.perspective_camera(dims, (96, 64), azimuth_deg=15.0)
    tf = wl.tf_src(28)
    a = sc.render_ea(M, 96, 64, 0.5, tf, bg=BG, tau=0.99)
    assert sc.ctx.get_plan(vr.MODE_EA)["skip_level"] == 3
    sc.ctx.set_option(vr.OPT_SKIP, 0)
    b = sc.render_ea(M, 96, 64, 0.5, tf, bg=BG, tau=0.99)
    assert np.array_equal(a, b)
