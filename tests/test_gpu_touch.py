"""vr_measure_touch / vr_touch_count (SURVEY.md 8(d) "B_touch"): the measurement pass bench.py's roofline rests on.

Pinned three ways: (1) a view whose footprints cover every stored voxel of every brick must set exactly the
sectors that the documented layout (re-typed here in numpy) assigns to those voxels;
(2) the pass must interpolate exactly the samples the production marchers report in their counters, at every
skipping level; (3) invariants: lines <= sectors <= 4 lines, a transparent table touches nothing, fewer
samples taken -> a subset of the sectors.
"""
import numpy as np
import pytest

from paper_1012_2909_b200 import workloads as wl

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def H():
    import helpers
    helpers.torch_cuda()
    helpers.FORCED_OPTIONS.clear()
    return helpers


def slot_layout1(lx, ly, lz, T0, T1):
    """Offset (floats) of stored voxel (lx, ly, lz) inside its brick: 4 x 4 x 2 micro-blocks of one 128-byte line."""
    return (32 * ((lx >> 2) + T0 * ((ly >> 2) + T1 * (lz >> 1))) + 16 * ((ly >> 1) & 1) + 8 * (lz & 1) + 4 * (ly & 1) + (lx & 3))


def touch(sc, mode, M, W, Hh, step, tf, tau):
    import torch
    sc.ctx.set_view(M, W, Hh, step)
    if tf is not None:
        sc.ctx.set_transfer_function(*tf)
    ids = sc.ctx.sort_bricks(mode)
    parts, n, nbytes = sc.ctx.partial_layout(mode, ids)
    arena = torch.zeros(max(nbytes, 16), dtype=torch.uint8, device="cuda")
    sc.vr.Context.bind_partials(parts, n, arena)
    bitmap = torch.empty(sc.ctx.touch_layout(), dtype=torch.uint8, device="cuda")
    sc.ctx.reset_counters()
    sc.ctx.render_bricks(mode, parts, n, tau)
    cnt = sc.ctx.get_counters()
    sc.ctx.measure_touch(mode, parts, n, bitmap, tau)
    t = sc.ctx.touch_count(bitmap)
    torch.cuda.synchronize()
    return t, cnt, bitmap.cpu().numpy(), ids


def test_every_stored_voxel_touched_by_a_covering_view(H):
    """Axis-aligned orthographic rays through every voxel centre, step 1/2, nothing skipped: the footprints
    (floor(p) and its +1 neighbours, the halo included) are all stored voxels l_a in [0, min(B_a, N_a - lo_a)]."""
    dims, brick = (21, 18, 13), (8, 8, 8)
    cube = (np.random.default_rng(3).normal(size=dims[::-1]) + 5.0).astype(np.float32)
    sc = H.Scene(dims, brick, cube=cube)
    sc.ctx.set_option(sc.vr.OPT_SKIP, 0)
    M, (W, Hh) = wl.axis_ortho_camera(dims, 2, +1)
    t, cnt, bits, ids = touch(sc, sc.vr.MODE_EA, M, W, Hh, 0.5, wl.tf_fog(), 2.0)
    assert t["taken_samples"] == cnt["taken_samples"] == cnt["nominal_samples"] > 0
    G = [-(-n // b) for n, b in zip(dims, brick)]
    T0, T1, T2 = (brick[0] + 1 + 3) // 4, (brick[1] + 1 + 3) // 4, (brick[2] + 1 + 1) // 2
    stride = 32 * T0 * T1 * T2
    want = np.zeros(bits.size * 8, dtype=bool)
    for bid in range(G[0] * G[1] * G[2]):
        b = (bid % G[0], (bid // G[0]) % G[1], bid // (G[0] * G[1]))
        hi = [min(brick[a], dims[a] - b[a] * brick[a]) for a in range(3)]
        lx, ly, lz = np.meshgrid(np.arange(hi[0] + 1), np.arange(hi[1] + 1), np.arange(hi[2] + 1), indexing="ij")
        # a brick whose first plane is the cube's last plane along an axis holds no sample (position N-1 belongs to it,
        # and is sampled: floor(N-1) = N-1), so it IS touched: its voxel l = 0 and the zero halo l = 1
        off = bid * stride + slot_layout1(lx, ly, lz, T0, T1)
        want[off.reshape(-1) >> 3] = True
    got = np.unpackbits(bits, bitorder="little").astype(bool)
    assert np.array_equal(got, want)
    assert t["sectors"] == int(want.sum())
    lines = want.reshape(-1, 4).any(axis=1).sum()
    assert t["lines"] == int(lines)


@pytest.mark.parametrize("variant,cell,occ", [(-1, -1, -1), (0, 1, 0), (0, 1, 1), (3, 1, 0), (3, 1, 1), (3, 0, 0)])
def test_taken_samples_equal_the_marchers_counters(H, variant, cell, occ):
    """The pass walks the samples one by one with the plan's exact tests, so for emission-absorption it interpolates
    the very samples the production marcher does (same skipping level, same ERT stop)."""
    w = wl.scaled(wl.C2, "touch", (96, 80, 112), (32, 32, 32), (200, 120), n_sources=12)
    sc = H.Scene(w.dims, w.brick, gen={"seed": w.seed, "sources": wl.make_sources(w)})
    vr = sc.vr
    sc.ctx.set_option(vr.OPT_VARIANT, variant)
    sc.ctx.set_option(vr.OPT_CELL_SKIP, cell)
    sc.ctx.set_option(vr.OPT_OCCUPANCY, occ)
    if variant == 3:
        sc.ctx.set_option(vr.OPT_DENSE, 0)
    M = wl.perspective_camera(w.dims, w.frame, azimuth_deg=40.0)
    W, Hh = w.frame
    tf = wl.tf_src(24)
    t, cnt, bits, _ = touch(sc, vr.MODE_EA, M, W, Hh, 0.5, tf, 0.9)
    assert t["taken_samples"] == cnt["taken_samples"] > 0
    assert t["lines"] <= t["sectors"] <= 4 * t["lines"]
    # nothing skipped, no ERT: every sample is taken and the sectors are a superset
    sc.ctx.set_option(vr.OPT_SKIP, 0)
    t_all, cnt_all, bits_all, _ = touch(sc, vr.MODE_EA, M, W, Hh, 0.5, tf, 2.0)
    assert t_all["taken_samples"] == cnt_all["nominal_samples"]
    assert (bits & ~bits_all).max() == 0 and t_all["sectors"] > t["sectors"]
    # MIP: the pass follows each ray in order (running maximum), the lockstep marcher tests a chunk of samples against a
    # slightly older maximum: it may take more, never fewer
    sc.ctx.set_option(vr.OPT_SKIP, 1)
    tm, cm, _, _ = touch(sc, vr.MODE_MIP, M, W, Hh, 0.5, None, 2.0)
    assert 0 < tm["taken_samples"] <= cm["taken_samples"] <= cm["nominal_samples"]


def test_transparent_table_touches_nothing(H):
    dims, brick = (40, 40, 40), (16, 16, 16)
    cube = np.random.default_rng(5).normal(size=dims[::-1]).astype(np.float32)
    sc = H.Scene(dims, brick, cube=cube)
    table = np.zeros((256, 4), dtype=np.float32)
    table[:, :3] = 0.5
    table[250:, 3] = 0.5                                  # only values above 31 are opaque: none in N(0,1)
    M = wl.perspective_camera(dims, (64, 48), azimuth_deg=10.0)
    import torch
    sc.ctx.set_view(M, 64, 48, 0.5)
    sc.ctx.set_transfer_function(table, 0.0, 32.0)
    ids = sc.ctx.sort_bricks(sc.vr.MODE_EA)
    assert len(ids) == 0                                   # every brick is inactive: nothing to render or to touch
    # force the bricks into the list: the finer levels must still reject every sample
    g = sc.grid()
    ids = np.arange(g[0] * g[1] * g[2], dtype=np.int32)
    parts, n, nbytes = sc.ctx.partial_layout(sc.vr.MODE_EA, ids)
    arena = torch.zeros(max(nbytes, 16), dtype=torch.uint8, device="cuda")
    sc.vr.Context.bind_partials(parts, n, arena)
    bitmap = torch.empty(sc.ctx.touch_layout(), dtype=torch.uint8, device="cuda")
    sc.ctx.measure_touch(sc.vr.MODE_EA, parts, n, bitmap, 0.99)
    t = sc.ctx.touch_count(bitmap)
    assert t == {"sectors": 0, "lines": 0, "taken_samples": 0}
