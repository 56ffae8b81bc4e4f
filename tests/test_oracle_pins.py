"""Pins of the CPU oracle (oracle/ovr.cpp) against what the mathematics fixes - closed forms,
invariants, special cases and brute force - as listed in SURVEY.md section 8(c), "What pins each
part".  CPU only.  None of these retypes the oracle's own formula as the expected value: each is
a different route to the same number (a column maximum, Beer-Lambert, an affine field, ...).
"""
import math

import numpy as np
import pytest

from paper_1012_2909_b200 import workloads as wl

BG = (0.25, 0.5, 0.125, 0.75)


def const_tf(rgb, a, vmin=0.0, vmax=1.0):
    t = np.zeros((256, 4), dtype=np.float32)
    t[:, :3] = rgb
    t[:, 3] = a
    return t, vmin, vmax


def noise_cube(shape, seed=0):
    return np.random.default_rng(seed).normal(size=shape).astype(np.float32)


def rand_persp(dims, frame, seed):
    rng = np.random.default_rng(seed)
    return wl.perspective_camera(dims, frame, azimuth_deg=rng.uniform(0, 360),
                                 elevation_deg=rng.uniform(-60, 60), fovy_deg=rng.uniform(20, 60))


# ------------------------------------------------------------------------------ paper sizes
def test_golden_paper_sizes():
    vals = {}
    import os
    with open(os.path.join(os.path.dirname(__file__), "golden", "paper_sizes.txt")) as f:
        for line in f:
            line = line.split("#")[0].split()
            if len(line) == 2:
                vals[line[0]] = float(line[1])
    assert vals["panel_cols"] * vals["panel_width"] == vals["wall_width"]
    assert vals["panel_rows"] * vals["panel_height"] == vals["wall_height"]
    # "12 GB" pins 4 bytes per voxel (float32), 2.2 TB likewise for the WALLABY cube
    gb = vals["hipass_nx"] * vals["hipass_ny"] * vals["hipass_nz"] * 4 / 1e9
    assert round(gb) == vals["hipass_gigabytes"]
    tib = vals["wallaby_nx"] * vals["wallaby_ny"] * vals["wallaby_nz"] * 4 / 2 ** 40
    assert abs(tib - vals["wallaby_terabytes"]) < 0.1
    for name in ("C4", "C5"):
        w = wl.CONFIGS[name]
        assert w.frame == (int(vals["wall_width"]), int(vals["wall_height"]))
        assert w.panels == (int(vals["panel_cols"]), int(vals["panel_rows"]))
        assert (w.frame[0] // w.panels[0], w.frame[1] // w.panels[1]) == (1920, 1080)


# ------------------------------------------------------------------------------ O-2 rays
def test_ray_invariants(ovr):
    dims, frame = (40, 30, 50), (37, 23)
    for seed in range(4):
        M = rand_persp(dims, frame, seed) if seed % 2 == 0 else \
            wl.ortho_camera(dims, frame, wl.seeded_directions(seed, 1)[0])
        M64 = M.astype(np.float64)
        for (i, j) in [(0, 0), (36, 22), (18, 11), (5, 20)]:
            o, d, L = ovr.ray(M, *frame, 0.5, i, j)
            assert abs(np.linalg.norm(d) - 1.0) < 1e-14
            xn, yn = 2 * (i + 0.5) / frame[0] - 1, 1 - 2 * (j + 0.5) / frame[1]
            for t in (0.0, 0.3 * L, L):
                c = M64 @ np.append(o + t * d, 1.0)
                assert abs(c[0] / c[3] - xn) < 1e-9 and abs(c[1] / c[3] - yn) < 1e-9
            zn0 = M64 @ np.append(o, 1.0)
            zn1 = M64 @ np.append(o + L * d, 1.0)
            assert abs(zn0[2] / zn0[3] + 1) < 1e-9 and abs(zn1[2] / zn1[3] - 1) < 1e-9


def test_axis_ortho_rays_hit_voxel_centres(ovr):
    dims = (12, 10, 8)
    for axis in range(3):
        for sign in (1, -1):
            M, (W, H) = wl.axis_ortho_camera(dims, axis, sign)
            ua, va = [(1, 2), (0, 2), (0, 1)][axis]
            assert W >= dims[ua] and H >= dims[va]
            for (i, j) in [(0, 0), (dims[ua] - 1, dims[va] - 1), (3, 2)]:
                o, d, L = ovr.ray(M, W, H, 0.5, i, j)
                assert o[ua] == i and o[va] == j           # exact: all values dyadic
                e = np.zeros(3); e[axis] = sign
                assert np.array_equal(d, e)
                assert o[axis] == (-8.0 if sign > 0 else dims[axis] - 1 + 8.0)


# ------------------------------------------------------------------------------ O-3 lattice
def test_lattice_count_axis_aligned(ovr):
    dims = (9, 7, 11)
    cube = noise_cube(dims[::-1])
    vol = ovr.Volume.linear(cube)
    for step in (0.5, 0.25, 1.0):
        for axis in range(3):
            M, (W, H) = wl.axis_ortho_camera(dims, axis, 1)
            _, _, c = ovr.render(vol, M, W, H, step, ovr.MIP, ovr.F64, brute=True)
            per_ray = math.floor((dims[axis] - 1) / step) + 1
            ua, va = [(1, 2), (0, 2), (0, 1)][axis]
            assert c["nominal"] == per_ray * dims[ua] * dims[va]


def test_bracket_equals_brute_force(ovr):
    dims, frame = (20, 17, 23), (24, 20)
    vol = ovr.Volume.linear(noise_cube(dims[::-1], 3))
    tf = wl.tf_ramp()
    for seed in range(3):
        M = rand_persp(dims, frame, 10 + seed)
        for prec in (ovr.F64, ovr.F32):
            a, _, ca = ovr.render(vol, M, *frame, 0.5, ovr.EA, prec, tf=tf, bg=BG, brute=True)
            b, _, cb = ovr.render(vol, M, *frame, 0.5, ovr.EA, prec, tf=tf, bg=BG, brute=False)
            assert np.array_equal(a, b) and ca == cb


# ------------------------------------------------------------------------------ O-4 trilinear
def affine_cube(dims, c):
    z, y, x = np.meshgrid(np.arange(dims[2]), np.arange(dims[1]), np.arange(dims[0]), indexing="ij")
    return (c[0] + c[1] * x + c[2] * y + c[3] * z).astype(np.float32)


def lattice_ends(ovr, M, W, H, step, dims, i, j):
    """First and last lattice positions inside the box, from the ray alone (fp64)."""
    o, d, L = ovr.ray(M, W, H, step, i, j)
    k = np.arange(0, int(L / step) + 1)
    p = o[None, :] + (k * step)[:, None] * d[None, :]
    ok = np.all((p >= 0) & (p <= np.array(dims) - 1), axis=1)
    if not ok.any():
        return None
    idx = np.nonzero(ok)[0]
    return p[idx[0]], p[idx[-1]]


def test_affine_field_mip_closed_form(ovr):
    # closed form 2: f affine => monotone along a ray => MIP = max(f(p_first), f(p_last));
    # pins trilinear (reproduces affine fields), perspective clipping and the lattice
    dims, frame = (24, 20, 28), (16, 12)
    c = (3.0, 0.5, -0.25, 0.125)
    vol = ovr.Volume.linear(affine_cube(dims, c))
    f = lambda p: c[0] + c[1] * p[0] + c[2] * p[1] + c[3] * p[2]
    for seed in range(3):
        M = rand_persp(dims, frame, 20 + seed)
        out, flags, _ = ovr.render(vol, M, *frame, 0.5, ovr.MIP, ovr.F64, miss=-99.0)
        checked = 0
        for j in range(frame[1]):
            for i in range(frame[0]):
                ends = lattice_ends(ovr, M, *frame, 0.5, dims, i, j)
                if flags[j, i]:
                    continue
                if ends is None:
                    assert out[j, i] == -99.0
                else:
                    assert abs(out[j, i] - max(f(ends[0]), f(ends[1]))) < 2e-5
                    checked += 1
        assert checked > 20


def test_trilinear_returns_voxels_and_is_bounded(ovr):
    # axis-aligned, step 1: every sample sits on a voxel centre => EA through a TF that is the
    # identity on alpha would be indirect; use MIP of -cube and +cube: both maxima are voxel values
    dims = (8, 8, 8)
    cube = noise_cube(dims[::-1], 5)
    vol = ovr.Volume.linear(cube)
    M, (W, H) = wl.axis_ortho_camera(dims, 2, 1)
    hi, _, _ = ovr.render(vol, M, W, H, 1.0, ovr.MIP, ovr.F32)
    lo, _, _ = ovr.render(ovr.Volume.linear(-cube), M, W, H, 1.0, ovr.MIP, ovr.F32)
    assert np.array_equal(hi[:8, :8], cube.max(axis=0)) and np.array_equal(-lo[:8, :8], cube.min(axis=0))
    # arbitrary views: interpolated maxima never exceed the cube maximum (and reach > min)
    for seed in range(3):
        Mp = rand_persp(dims, (20, 20), seed)
        m, _, _ = ovr.render(vol, Mp, 20, 20, 0.5, ovr.MIP, ovr.F32, miss=0.0)
        assert m.max() <= cube.max() and m.min() >= min(cube.min(), 0.0)


# ------------------------------------------------------------------------------ O-5 MIP
def test_mip_column_maximum_bit_exact(ovr):
    # closed form 1 (north_star: "axis-aligned orthographic MIP equal to the per-column maximum")
    dims = (13, 9, 17)
    cube = noise_cube(dims[::-1], 7)
    cube[-1, -1, -1] = 50.0          # maximum on the last voxel planes (O-4 clamp-duplicate rule)
    vol = ovr.Volume.linear(cube)
    for axis in range(3):
        for sign in (1, -1):
            M, (W, H) = wl.axis_ortho_camera(dims, axis, sign)
            for prec in (ovr.F32, ovr.F64):
                out, _, _ = ovr.render(vol, M, W, H, 0.5, ovr.MIP, prec, miss=-1.0)
                ua, va = [(1, 2), (0, 2), (0, 1)][axis]
                assert np.array_equal(out[:dims[va], :dims[ua]], cube.max(axis=2 - axis))
                assert (out[dims[va]:] == -1.0).all() and (out[:, dims[ua]:] == -1.0).all()


# ------------------------------------------------------------------------------ O-6 TF
def test_tf_entries_and_opacity_correction(ovr):
    tf = wl.tf_ramp()
    table, vmin, vmax = tf
    for step in (0.5, 0.25, 1.0):
        baked = ovr.bake_tf(tf, step)
        assert np.array_equal(baked[:, :3], table[:, :3])
        # (1 - a')^(1/step) = 1 - a
        assert np.allclose((1.0 - baked[:, 3].astype(np.float64)) ** (1.0 / step),
                           1.0 - table[:, 3].astype(np.float64), atol=1e-6)
        for i in (0, 1, 17, 128, 254, 255):
            v = vmin + i * (vmax - vmin) / 255.0
            q = ovr.tf_lookup(tf, step, v, baked=False)
            assert np.allclose(q, table[i], atol=1e-6)
        # ramp: colour r(v) = (v - vmin)/(vmax - vmin) analytically, also between entries
        for v in (0.37, 7.77, 19.2):
            q = ovr.tf_lookup(tf, step, v, baked=False)
            assert abs(q[0] - v / 20.0) < 1e-6 and abs(q[2] - (1 - v / 20.0)) < 1e-6
        # clamping outside [vmin, vmax]
        assert np.allclose(ovr.tf_lookup(tf, step, -5.0, baked=False), table[0], atol=1e-7)
        assert np.allclose(ovr.tf_lookup(tf, step, 50.0, baked=False), table[255], atol=1e-7)


# ------------------------------------------------------------------------------ O-7 EA
@pytest.mark.parametrize("prec_name", ["F64", "F32"])
def test_beer_lambert_constant_cube(ovr, prec_name):
    # north_star closed form: "Beer-Lambert emission-absorption through a constant-density cube"
    prec = getattr(ovr, prec_name)
    dims, step, a = (16, 16, 16), 0.5, 0.2
    rgb = np.array([0.9, 0.4, 0.1])
    vol = ovr.Volume.linear(np.full(dims[::-1], 0.5, dtype=np.float32))
    tf = const_tf(rgb, a)
    M, (W, H) = wl.axis_ortho_camera(dims, 2, 1)
    out, _, c = ovr.render(vol, M, W, H, step, ovr.EA, prec, tf=tf, tau=2.0)
    n = math.floor((dims[2] - 1) / step) + 1
    ap = 1.0 - (1.0 - a) ** step
    A = 1.0 - (1.0 - ap) ** n
    tol = 1e-6 if prec == ovr.F64 else 1e-5
    assert np.allclose(out[..., 3], A, atol=tol)
    assert np.allclose(out[..., :3], rgb * A, atol=tol)
    # continuous Beer-Lambert: (1-a')^n = exp(-kappa n step), |n step - L_box| < step
    kappa, Lbox = -math.log(1.0 - a), dims[2] - 1
    assert abs((1.0 - A) - math.exp(-kappa * Lbox)) <= kappa * step * math.exp(-kappa * Lbox) * 1.01
    # an oblique ray: n from the oracle's own counter is not used; use the ray geometry instead
    Mp = wl.perspective_camera(dims, (9, 9), azimuth_deg=33.0, elevation_deg=15.0)
    outp, flags, _ = ovr.render(vol, Mp, 9, 9, step, ovr.EA, prec, tf=tf, tau=2.0)
    for (i, j) in [(4, 4), (3, 5), (5, 3)]:
        ends = lattice_ends(ovr, Mp, 9, 9, step, dims, i, j)
        if ends is None or flags[j, i]:
            continue
        n_ij = int(round(np.linalg.norm(ends[1] - ends[0]) / step)) + 1
        A_ij = 1.0 - (1.0 - ap) ** n_ij
        assert abs(outp[j, i, 3] - A_ij) < tol * 3


def test_two_slab_front_to_back_order(ovr):
    # two constant halves along z, axis-aligned: closed form; the opposite view mirrors it
    dims, step = (8, 8, 16), 1.0            # step 1: samples on voxel centres only
    cube = np.zeros(dims[::-1], dtype=np.float32)
    cube[:8] = 0.0       # z < 8  -> TF entry 0
    cube[8:] = 1.0       # z >= 8 -> TF entry 255
    t = np.zeros((256, 4), dtype=np.float32)
    t[0] = (1.0, 0.0, 0.0, 0.3)
    t[255] = (0.0, 0.0, 1.0, 0.6)
    for i in range(1, 255):                 # unused in-between entries (values are exactly 0 or 1)
        t[i] = t[0] + (t[255] - t[0]) * i / 255.0
    tf = (t, 0.0, 1.0)
    vol = ovr.Volume.linear(cube)

    def slab(a, n):                          # n samples of opacity a: (colour weight, alpha)
        A = 1.0 - (1.0 - a) ** n
        return A

    A1, A2 = slab(0.3, 8), slab(0.6, 8)
    front_red = np.array([A1, 0.0, (1 - A1) * A2, A1 + (1 - A1) * A2])
    front_blue = np.array([(1 - A2) * A1, 0.0, A2, A2 + (1 - A2) * A1])
    M, (W, H) = wl.axis_ortho_camera(dims, 2, +1)
    out, _, _ = ovr.render(vol, M, W, H, step, ovr.EA, ovr.F64, tf=tf)
    assert np.allclose(out, front_red, atol=1e-6)
    M, (W, H) = wl.axis_ortho_camera(dims, 2, -1)
    out2, _, _ = ovr.render(vol, M, W, H, step, ovr.EA, ovr.F64, tf=tf)
    assert np.allclose(out2, front_blue, atol=1e-6)
    assert np.abs(out - out2).max() > 0.1    # order matters


def test_ert_stop_step_and_bound(ovr):
    dims, step, a, tau = (8, 8, 64), 0.5, 0.15, 0.9
    rgb = np.array([0.2, 0.7, 0.5])
    vol = ovr.Volume.linear(np.full(dims[::-1], 0.5, dtype=np.float32))
    tf = const_tf(rgb, a)
    M, (W, H) = wl.axis_ortho_camera(dims, 2, 1)
    out, _, c = ovr.render(vol, M, W, H, step, ovr.EA, ovr.F64, tf=tf, tau=tau)
    full, _, cf = ovr.render(vol, M, W, H, step, ovr.EA, ovr.F64, tf=tf, tau=2.0)
    ap = 1.0 - (1.0 - a) ** step
    nstar = math.ceil(math.log(1.0 - tau) / math.log(1.0 - ap))
    assert (W, H) == (8, 8)
    assert c["taken"] == nstar * W * H and c["terminated"] == W * H
    assert cf["taken"] == cf["nominal"] and cf["terminated"] == 0
    A = out[..., 3]
    assert (A >= tau).all() and (A <= tau + (1 - tau) * ap + 1e-7).all()
    assert np.abs(out - full).max() <= (1 - tau) / tau


def test_empty_cube_renders_background(ovr):
    # north_star closed form: "an empty cube rendering to the background colour"
    dims = (10, 10, 10)
    vol = ovr.Volume.linear(np.zeros(dims[::-1], dtype=np.float32))
    tf = wl.tf_src()                          # a(0) = 0
    M = wl.perspective_camera(dims, (21, 17))
    for prec in (ovr.F32, ovr.F64):
        out, _, _ = ovr.render(vol, M, 21, 17, 0.5, ovr.EA, prec, tf=tf, bg=BG, tau=0.99)
        assert np.array_equal(out, np.broadcast_to(np.array(BG, dtype=np.float32), out.shape))
        mip, _, c = ovr.render(vol, M, 21, 17, 0.5, ovr.MIP, prec, miss=-7.0)
        assert set(np.unique(mip)) <= {0.0, -7.0} and (mip == 0.0).any() and (mip == -7.0).any()


# ------------------------------------------------------------------------------ O-8 / O-9 bricks
@pytest.mark.parametrize("persp", [True, False])
def test_brick_split_equals_unsplit(ovr, persp):
    # north_star closed form: "compositing of any brick split equal to the unsplit render"
    dims, frame = (20, 16, 24), (22, 18)
    cube = np.abs(noise_cube(dims[::-1], 11)) * 4.0
    vol = ovr.Volume.linear(cube)
    tf = wl.tf_fog()
    for seed in range(3):
        M = rand_persp(dims, frame, 30 + seed) if persp else \
            wl.ortho_camera(dims, frame, wl.seeded_directions(40 + seed, 1)[0])
        for part in [(8, 8, 8), (5, 16, 7), (20, 16, 24), (3, 3, 3)]:
            # MIP: exactly associative and commutative -> bit-exact in both split modes
            ref, _, c0 = ovr.render(vol, M, *frame, 0.5, ovr.MIP, ovr.F32)
            for split in (ovr.SPLIT_GLOBAL, ovr.SPLIT_SORTLAST):
                got, _, c1 = ovr.render(vol, M, *frame, 0.5, ovr.MIP, ovr.F32, split=split, partition=part)
                assert np.array_equal(ref, got) and c0["nominal"] == c1["taken"]
            # EA, GLOBAL accumulator: bit-exact in float32 arithmetic, any tau
            for tau in (0.9, 2.0):
                ref, _, c0 = ovr.render(vol, M, *frame, 0.5, ovr.EA, ovr.F32, tf=tf, bg=BG, tau=tau)
                got, _, c1 = ovr.render(vol, M, *frame, 0.5, ovr.EA, ovr.F32, tf=tf, bg=BG, tau=tau,
                                        split=ovr.SPLIT_GLOBAL, partition=part)
                assert np.array_equal(ref, got) and c0 == c1
            # EA, sort-last, ERT disabled: equal up to fp reassociation
            ref, _, _ = ovr.render(vol, M, *frame, 0.5, ovr.EA, ovr.F64, tf=tf, bg=BG, tau=2.0)
            got, _, _ = ovr.render(vol, M, *frame, 0.5, ovr.EA, ovr.F64, tf=tf, bg=BG, tau=2.0,
                                   split=ovr.SPLIT_SORTLAST, partition=part)
            assert np.abs(ref - got).max() < 1e-6
            # EA, sort-last, local ERT: bounded by (1 - tau) / tau
            got, _, _ = ovr.render(vol, M, *frame, 0.5, ovr.EA, ovr.F64, tf=tf, bg=BG, tau=0.9,
                                   split=ovr.SPLIT_SORTLAST, partition=part)
            assert np.abs(ref - got).max() <= 0.1 / 0.9 + 1e-6


def test_partials_plus_composite_equal_sortlast_render(ovr):
    dims, frame, part = (16, 16, 16), (20, 20), (8, 8, 8)
    cube = np.abs(noise_cube(dims[::-1], 13)) * 4.0
    vol = ovr.Volume.linear(cube)
    tf = wl.tf_fog()
    M = rand_persp(dims, frame, 50)
    keys, persp = ovr.visibility_keys(M, *frame, 0.5, part, (2, 2, 2))
    order = ovr.visibility_order(keys)
    full = (0, 0, frame[0], frame[1])
    for mode in (ovr.EA, ovr.MIP):
        partials = [ovr.render_brick(vol, M, *frame, 0.5, mode, b, full, part, ovr.F32, tf=tf, tau=0.95)
                    for b in range(8)]
        got = ovr.composite(mode, [full] * 8, partials, order, *frame, bg=BG, miss=-1.0, precision=ovr.F32)
        ref, _, _ = ovr.render(vol, M, *frame, 0.5, mode, ovr.F32, tf=tf, bg=BG, tau=0.95, miss=-1.0,
                               split=ovr.SPLIT_SORTLAST, partition=part)
        assert np.array_equal(got, ref)
        if mode == ovr.EA:
            # a fully transparent partial is the identity; reversing the order changes the frame
            zero = np.zeros_like(partials[0])
            got2 = ovr.composite(mode, [full] * 9, partials + [zero], list(order[:3]) + [8] + list(order[3:]),
                                 *frame, bg=BG, precision=ovr.F32)
            assert np.array_equal(got2, ref)
            rev = ovr.composite(mode, [full] * 8, partials, order[::-1], *frame, bg=BG, precision=ovr.F32)
            assert np.abs(rev - ref).max() > 1e-3


def test_visibility_keys_brute_force(ovr):
    # O-9: along every ray the key must strictly increase from brick to brick
    rng = np.random.default_rng(5)
    for grid, brick in [((2, 2, 2), (4, 4, 4)), ((3, 3, 3), (3, 3, 3)), ((3, 4, 2), (4, 3, 5))]:
        dims = tuple(g * b for g, b in zip(grid, brick))
        frame = (15, 13)
        cams = [rand_persp(dims, frame, s) for s in range(6)]
        cams += [wl.ortho_camera(dims, frame, d) for d in wl.seeded_directions(9, 4)]
        cams += [wl.ortho_camera(dims, frame, d) for d in ([1, 0, 0], [0, -1, 0], [0, 1, 1], [1, 0, -1])]
        # eye inside the grid / on a brick plane
        c = (np.array(dims) - 1) / 2.0
        for eye in (c + 0.3, np.array([brick[0], c[1], c[2]], dtype=float)):
            V = wl._look_at(eye, eye + np.array([0.3, 0.2, 1.0]), np.array([0.0, 1.0, 0.0]))
            cams.append((wl._frustum(-0.5, 0.5, -0.5, 0.5, 0.5, 200.0) @ V).astype(np.float32))
        for M in cams:
            keys, _ = ovr.visibility_keys(M, *frame, 0.25, brick, grid)
            for j in range(0, frame[1], 2):
                for i in range(0, frame[0], 2):
                    o, d, L = ovr.ray(M, *frame, 0.25, i, j)
                    t = np.arange(0, L, 0.05)
                    p = o[None] + t[:, None] * d[None]
                    ok = np.all((p >= 0) & (p <= np.array(dims) - 1), axis=1)
                    b = (np.floor(p[ok]) // np.array(brick)).astype(int)
                    ids = b[:, 0] + grid[0] * (b[:, 1] + grid[1] * b[:, 2])
                    seq = ids[np.insert(np.diff(ids) != 0, 0, True)] if len(ids) else ids
                    k = keys[seq]
                    assert (np.diff(k) > 0).all(), (grid, i, j, seq, k)


# ------------------------------------------------------------------------------ S6 tiled frame
def test_tiled_panels_equal_single_frustum(ovr):
    dims = (24, 24, 32)
    cube = np.abs(noise_cube(dims[::-1], 17)) * 3.0
    vol = ovr.Volume.linear(cube)
    tf = wl.tf_fog()
    cols, rows, pw, ph = 5, 5, 8, 6
    W, H = cols * pw, rows * ph
    M = wl.perspective_camera(dims, (W, H))
    ref, _, _ = ovr.render(vol, M, W, H, 0.5, ovr.EA, ovr.F64, tf=tf, bg=BG)
    tiled = np.zeros_like(ref)
    for r in range(rows):
        for c in range(cols):
            Mp = wl.panel_matrix(M, cols, rows, c, r)
            out, _, _ = ovr.render(vol, Mp, pw, ph, 0.5, ovr.EA, ovr.F64, tf=tf, bg=BG)
            tiled[r * ph:(r + 1) * ph, c * pw:(c + 1) * pw] = out
    # identical rays up to the float32 rounding of the panel matrices
    assert np.abs(ref - tiled).max() < 1e-4


# ------------------------------------------------------------------------------ O-11 precision
def test_float32_arithmetic_within_tolerance_of_float64(ovr):
    dims, frame = (48, 40, 56), (40, 30)
    w = wl.scaled(wl.C2, "t", dims, (16, 16, 16), frame, n_sources=6)
    cube = ovr.generate(w.seed, dims, sources=wl.make_sources(w))
    vol = ovr.Volume.linear(cube)
    tf = wl.tf_fog()
    M = wl.perspective_camera(dims, frame)
    a, fl, _ = ovr.render(vol, M, *frame, 0.5, ovr.EA, ovr.F64, tf=tf, tau=0.99)
    b, _, _ = ovr.render(vol, M, *frame, 0.5, ovr.EA, ovr.F32, tf=tf, tau=0.99)
    ok = fl == 0
    assert ok.mean() > 0.99
    err = np.abs(a - b)[ok]
    assert err.max() <= 1e-4 and math.sqrt((err ** 2).mean()) <= 1e-5


# ------------------------------------------------------------------------------ generator
def test_noise_statistics(ovr):
    n = 200000
    x = np.array([ovr.noise(1234, i) for i in range(n)])
    assert abs(x.mean()) < 4 / math.sqrt(n) and abs(x.std() - 1) < 0.01
    # Kolmogorov-Smirnov against N(0,1)
    xs = np.sort(x)
    cdf = 0.5 * (1 + np.array([math.erf(v / math.sqrt(2)) for v in xs]))
    D = np.max(np.abs(cdf - (np.arange(1, n + 1) - 0.5) / n))
    assert D < 1.63 / math.sqrt(n)
    assert abs(np.corrcoef(x[:-1], x[1:])[0, 1]) < 0.01
    assert ovr.noise(1234, 5) != ovr.noise(1235, 5)


def test_generator_sources_and_determinism(ovr):
    w = wl.scaled(wl.C2, "t", (96, 80, 128), (32, 32, 32), (64, 64), n_sources=5)
    S = wl.make_sources(w)
    full = ovr.generate(w.seed, w.dims, sources=S)
    noise_only = ovr.generate(w.seed, w.dims)
    sig = full.astype(np.float64) - noise_only
    assert abs(noise_only.std() - 1) < 0.01
    # each source: the signal at the voxel nearest its centre is close to its amplitude, and the
    # signal vanishes outside the union of bounding boxes
    for s in S:
        c = np.rint(s[:3]).astype(int)
        lone = ovr.generate(w.seed, w.dims, region=(c[0], c[1], c[2], 1, 1, 1), sources=s[None])[0, 0, 0] \
            - noise_only[c[2], c[1], c[0]]
        d = c - s[:3]
        assert lone <= s[wl.S_AMP] + 1e-5 and lone > s[wl.S_AMP] * math.exp(-0.5 * 3 * 0.25 / min(s[wl.S_SA], s[wl.S_SB], s[wl.S_SZ]) ** 2 * 4) - 1e-4
    mask = np.zeros(full.shape, dtype=bool)
    for s in S:
        b = s[wl.S_XLO:].astype(int)
        mask[b[4]:b[5] + 1, b[2]:b[3] + 1, b[0]:b[1] + 1] = True
    assert np.abs(sig[~mask]).max() < 1e-6 and np.abs(sig[mask]).max() > 2.0
    # determinism, and independence of the generated region
    again = ovr.generate(w.seed, w.dims, sources=S)
    assert np.array_equal(full, again)
    reg = ovr.generate(w.seed, w.dims, region=(10, 7, 20, 33, 21, 40), sources=S)
    assert np.array_equal(reg, full[20:60, 7:28, 10:43])
    # continuum ramp and zero boxes
    ramp = ovr.generate(w.seed, w.dims, continuum=2.0)
    assert np.allclose(ramp[-1] - noise_only[-1], 2.0, atol=1e-6) and np.allclose(ramp[0], noise_only[0])
    zb = np.array([[0, 31, 32, 63, 64, 95]], dtype=np.int32)
    z = ovr.generate(w.seed, w.dims, sources=S, zero_boxes=zb)
    assert (z[64:96, 32:64, 0:32] == 0).all() and np.array_equal(z[:64], full[:64])


# ------------------------------------------------------------------ O-14 catalogue overlay
def _brute_edge_points(M, W, H, box, per_edge=6000):
    """Independent of the oracle's DDA: dense points along the 12 edges of a box in 3-D, kept where
    the clip-space point is inside near/far, projected to pixel coordinates (numpy fp64)."""
    M = np.asarray(M, dtype=np.float64).reshape(4, 4)
    xs, ys, zs = (box[0], box[1]), (box[2], box[3]), (box[4], box[5])
    pts = []
    t = np.linspace(0.0, 1.0, per_edge)[:, None]
    for a in range(3):
        for c in range(4):
            lo, hi = [0, 0, 0], [0, 0, 0]
            a1, a2 = (a + 1) % 3, (a + 2) % 3
            rng = (xs, ys, zs)
            lo[a], hi[a] = rng[a]
            lo[a1] = hi[a1] = rng[a1][c & 1]
            lo[a2] = hi[a2] = rng[a2][(c >> 1) & 1]
            p = np.array(lo, float)[None] * (1 - t) + np.array(hi, float)[None] * t
            clip = np.c_[p, np.ones(len(p))] @ M.T
            ok = (clip[:, 3] > 1e-9) & (np.abs(clip[:, 2]) <= clip[:, 3])
            clip = clip[ok]
            if len(clip):
                px = (clip[:, 0] / clip[:, 3] + 1) * 0.5 * W - 0.5
                py = (1 - clip[:, 1] / clip[:, 3]) * 0.5 * H - 0.5
                pts.append(np.c_[px, py])
    return np.concatenate(pts) if pts else np.zeros((0, 2))


def _check_against_brute(pick, pts, ident):
    H, W = pick.shape
    drawn = np.argwhere(pick == ident)[:, ::-1].astype(np.float64)         # (x, y)
    inside = pts[(pts[:, 0] > -0.49) & (pts[:, 0] < W - 0.51) & (pts[:, 1] > -0.49) & (pts[:, 1] < H - 0.51)]
    assert len(drawn) > 0 and len(inside) > 0
    # every drawn pixel hugs an edge: within half a pixel diagonal (+ the brute sampling pitch)
    d = np.sqrt(((drawn[:, None, :] - inside[None, ::7, :]) ** 2).sum(-1)).min(axis=1)
    assert d.max() <= 0.5 * np.sqrt(2.0) + 0.2, d.max()
    # no gaps: the DDA steps the major axis by <= 1, so a point of an edge is within 1/2 (along the
    # major axis) of a sample, whose pixel is within 1/2 per axis of it: sqrt(1 + 1/4).  Points closer
    # than a pixel to the viewport border are left out (their sample may round outside).
    sub = inside[(inside[:, 0] > 0.5) & (inside[:, 0] < W - 1.5) & (inside[:, 1] > 0.5) & (inside[:, 1] < H - 1.5)][::11]
    d2 = np.sqrt(((sub[:, None, :] - drawn[None, :, :]) ** 2).sum(-1)).min(axis=1)
    assert d2.max() <= math.sqrt(1.25) + 1e-9, d2.max()


def test_overlay_axis_view_draws_exact_rectangles(ovr):
    dims = (48, 40, 56)
    M, (W, H) = wl.axis_ortho_camera(dims, axis=2, sign=+1)
    boxes = np.array([[5, 20, 7, 30, 3, 50], [25, 25, 10, 12, 0, 55]], dtype=np.int32)    # the 2nd is 1 voxel wide
    pick = ovr.overlay(M, W, H, boxes)
    want = np.zeros((H, W), dtype=np.int32)
    for b, (x0, x1, y0, y1, _, _) in enumerate(boxes):
        want[y0, x0:x1 + 1] = np.maximum(want[y0, x0:x1 + 1], b + 1)
        want[y1, x0:x1 + 1] = np.maximum(want[y1, x0:x1 + 1], b + 1)
        want[y0:y1 + 1, x0] = np.maximum(want[y0:y1 + 1, x0], b + 1)
        want[y0:y1 + 1, x1] = np.maximum(want[y0:y1 + 1, x1], b + 1)
    assert np.array_equal(pick, want)


@pytest.mark.parametrize("az", [10.0, 135.0])
def test_overlay_perspective_hugs_projected_edges(ovr, az):
    dims = (96, 80, 160)
    W, H = 320, 180
    M = wl.perspective_camera(dims, (W, H), azimuth_deg=az)
    boxes = np.array([[10, 40, 12, 30, 20, 90], [50, 90, 40, 75, 100, 150]], dtype=np.int32)
    for b in range(2):
        vis = np.zeros(2, np.uint8)
        vis[b] = 1
        pick = ovr.overlay(M, W, H, boxes, vis)
        assert set(np.unique(pick)) == {0, b + 1}
        _check_against_brute(pick, _brute_edge_points(M, W, H, boxes[b]), b + 1)


def test_overlay_clips_at_the_near_plane(ovr):
    dims = (64, 64, 64)
    W, H = 200, 120
    # eye inside the cube looking along +z: boxes behind the eye vanish, a box around the eye is clipped
    eye = np.array([31.5, 31.5, 20.0])
    V = wl._look_at(eye, eye + np.array([0.0, 0.0, 1.0]), np.array([0.0, 1.0, 0.0]))
    top = 0.5 * math.tan(math.radians(30.0))
    M = (wl._frustum(-top * W / H, top * W / H, -top, top, 0.5, 200.0) @ V).astype(np.float32)
    behind = np.array([[10, 50, 10, 50, 0, 15]], dtype=np.int32)
    assert not ovr.overlay(M, W, H, behind).any()
    straddle = np.array([[20, 44, 22, 40, 5, 45]], dtype=np.int32)
    pick = ovr.overlay(M, W, H, straddle)
    _check_against_brute(pick, _brute_edge_points(M, W, H, straddle[0], per_edge=40000), 1)


def test_overlay_priority_visibility_and_pick(ovr):
    dims = (64, 64, 64)
    M, (W, H) = wl.axis_ortho_camera(dims, axis=2, sign=+1)
    boxes = np.array([[10, 30, 10, 30, 0, 10], [20, 40, 20, 40, 0, 10]], dtype=np.int32)
    both = ovr.overlay(M, W, H, boxes)
    assert both[20, 30] == 2 and both[30, 20] == 2          # crossings of the two outlines: the higher id wins
    only0 = ovr.overlay(M, W, H, boxes, np.array([1, 0], np.uint8))
    assert only0[20, 30] == 1 and only0[30, 20] == 1 and not (only0 == 2).any()
    assert not ovr.overlay(M, W, H, boxes, np.zeros(2, np.uint8)).any()
    assert np.array_equal(ovr.overlay(M, W, H, boxes, np.ones(2, np.uint8)), both)
    # pick: nearest covered pixel, ties to the larger id, -1 when nothing is near
    assert ovr.overlay_pick(both, 12, 15, 3) == 0            # 2 px right of box 0's left side
    assert ovr.overlay_pick(both, 38, 35, 3) == 1
    assert ovr.overlay_pick(both, 25, 25, 3) == -1           # inside both outlines, 5 px from any edge
    assert ovr.overlay_pick(both, 25, 25, 5) == 1            # box 0's side x=30 and box 1's side x=20 both at 5: tie
    assert ovr.overlay_pick(both, 60, 60, 4) == -1
    colours = np.array([[1, 0, 0, 1], [0, 1, 0, 1]], np.float32)
    frame = ovr.overlay_apply(np.full((H, W, 4), 0.25, np.float32), both, colours)
    assert np.array_equal(frame[10, 15], colours[0]) and np.array_equal(frame[20, 30], colours[1])
    assert np.array_equal(frame[0, 0], np.full(4, 0.25, np.float32))
