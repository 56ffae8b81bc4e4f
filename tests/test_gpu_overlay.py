"""NEXT-2: catalogue overlay on the GPU against the oracle (O-14; PAPER.md lines
31-33 section 2).  The catalogue is synthetic: the integer bounding boxes of the generator's own
seeded sources (the paper's Duchamp files are not in the container).  Integer output: bit-exact."""
import math

import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def _catalogue(wl, w):
    src = wl.make_sources(w)
    boxes = src[:, wl.S_XLO:wl.S_ZHI + 1].astype(np.int32)
    rng = np.random.default_rng(w.seed)
    colours = rng.uniform(0.0, 1.0, (len(boxes), 4)).astype(np.float32)
    colours[:, 3] = 1.0
    return boxes, colours


def _gpu_overlay(torch, ctx, boxes, colours, visible, frame, W, H, x0=0, y0=0, pick=None):
    d_boxes = torch.from_numpy(boxes).cuda()
    d_col = torch.from_numpy(colours).cuda() if colours is not None else None
    d_vis = torch.from_numpy(visible).cuda() if visible is not None else None
    if pick is None:
        pick = torch.full((H, W), -9, dtype=torch.int32, device="cuda")
    ctx.overlay_catalogue(d_boxes, d_col, d_vis, frame, pick)
    torch.cuda.synchronize()
    return pick


@pytest.mark.parametrize("az", [0.0, 35.0, 200.0])
def test_overlay_matches_oracle_bit_for_bit(az):
    import torch
    from paper_1012_2909_b200 import vr, workloads as wl
    from oracle import ovr
    w = wl.scaled(wl.C2, "ovl", (128, 128, 256), (64, 64, 64), (480, 270), n_sources=60)
    boxes, colours = _catalogue(wl, w)
    W, H = w.frame
    M = wl.perspective_camera(w.dims, w.frame, azimuth_deg=az)
    ctx = vr.Context(0)
    ctx.set_view(M, W, H, 0.5)
    vis = (np.arange(len(boxes)) % 3 != 0).astype(np.uint8)
    frame = torch.full((H, W, 4), 0.125, dtype=torch.float32, device="cuda")
    pick = _gpu_overlay(torch, ctx, boxes, colours, vis, frame, W, H).cpu().numpy()
    want = ovr.overlay(M, W, H, boxes, vis)
    assert want.any()
    assert np.array_equal(pick, want)
    assert np.array_equal(frame.cpu().numpy(), ovr.overlay_apply(np.full((H, W, 4), 0.125, np.float32), want, colours))
    # all shown, no frame painted
    pick2 = _gpu_overlay(torch, ctx, boxes, None, None, None, W, H).cpu().numpy()
    assert np.array_equal(pick2, ovr.overlay(M, W, H, boxes))
    # pick: a grid of clicks
    d_pick = torch.from_numpy(want).cuda()
    for (x, y, r) in [(10, 10, 4), (W // 2, H // 2, 6), (W // 3, H // 2, 2), (W - 1, H - 1, 8), (200, 100, 0), (240, 135, 64)]:
        assert ctx.overlay_pick(d_pick, x, y, r) == ovr.overlay_pick(want, x, y, r)


def test_overlay_near_plane_axis_views_and_empty_catalogue():
    import torch
    from paper_1012_2909_b200 import vr, workloads as wl
    from oracle import ovr
    dims = (64, 64, 64)
    W, H = 200, 120
    eye = np.array([31.5, 31.5, 20.0])
    V = wl._look_at(eye, eye + np.array([0.0, 0.0, 1.0]), np.array([0.0, 1.0, 0.0]))
    top = 0.5 * math.tan(math.radians(30.0))
    M = (wl._frustum(-top * W / H, top * W / H, -top, top, 0.5, 200.0) @ V).astype(np.float32)
    boxes = np.array([[10, 50, 10, 50, 0, 15], [20, 44, 22, 40, 5, 45], [0, 63, 0, 63, 0, 63], [30, 33, 30, 33, 21, 22]], dtype=np.int32)
    ctx = vr.Context(0)
    ctx.set_view(M, W, H, 0.5)
    pick = _gpu_overlay(torch, ctx, boxes, None, None, None, W, H).cpu().numpy()
    assert np.array_equal(pick, ovr.overlay(M, W, H, boxes))
    Ma, (Wa, Ha) = wl.axis_ortho_camera(dims, axis=1, sign=-1)
    ctx.set_view(Ma, Wa, Ha, 0.5)
    pick = _gpu_overlay(torch, ctx, boxes, None, None, None, Wa, Ha).cpu().numpy()
    want = ovr.overlay(Ma, Wa, Ha, boxes)
    assert want.any() and np.array_equal(pick, want)
    # empty catalogue: the viewport of the pick image is cleared, nothing else happens
    empty = _gpu_overlay(torch, ctx, np.zeros((0, 6), np.int32), None, None, None, Wa, Ha).cpu().numpy()
    assert not empty.any()


def test_overlay_on_tiled_panels_equals_single_frustum():
    """the 5 x 5 panels of one camera: the wireframes drawn panel by panel into one pitched
    frame are the oracle's panel images side by side."""
    import torch
    from paper_1012_2909_b200 import vr, workloads as wl
    from oracle import ovr
    w = wl.scaled(wl.C4, "ovlp", (96, 96, 192), (32, 32, 32), (400, 225), n_sources=30, panels=(5, 5))
    boxes, colours = _catalogue(wl, w)
    W, H = w.frame
    pw, ph = W // 5, H // 5
    M = wl.perspective_camera(w.dims, w.frame, azimuth_deg=30.0)
    ctx = vr.Context(0)
    pick = torch.full((H, W), -9, dtype=torch.int32, device="cuda")
    frame = torch.zeros((H, W, 4), dtype=torch.float32, device="cuda")
    want = np.zeros((H, W), np.int32)
    for r in range(5):
        for c in range(5):
            Mp = wl.panel_matrix(M, 5, 5, c, r)
            ctx.set_view(Mp, pw, ph, w.step)
            ctx.set_viewport(c * pw, r * ph, W)
            _gpu_overlay(torch, ctx, boxes, colours, None, frame, pw, ph, pick=pick)
            want[r * ph:(r + 1) * ph, c * pw:(c + 1) * pw] = ovr.overlay(Mp, pw, ph, boxes)
    got = pick.cpu().numpy()
    assert np.array_equal(got, want)
    assert np.array_equal(frame.cpu().numpy(), ovr.overlay_apply(np.zeros((H, W, 4), np.float32), want, colours))
    # the panels' wireframes continue across the seams: almost every pixel of the single-frustum
    # image is within one pixel of a panel-drawn pixel (the sampling phase differs per panel)
    whole = ovr.overlay(M, W, H, boxes) > 0
    ys, xs = np.nonzero(whole)
    near = np.zeros_like(whole)
    g = got > 0
    for dy in (-1, 0, 1):
        for dx in (-1, 0, 1):
            near |= np.roll(np.roll(g, dy, 0), dx, 1)
    assert near[ys, xs].mean() > 0.995


def test_overlay_error_codes():
    import torch
    from paper_1012_2909_b200 import vr
    ctx = vr.Context(0)
    pick = torch.zeros((4, 4), dtype=torch.int32, device="cuda")
    boxes = torch.zeros((1, 6), dtype=torch.int32, device="cuda")
    with pytest.raises(vr.VRError) as e:
        ctx.overlay_catalogue(boxes, None, None, None, pick)
    assert e.value.status == vr.ERR_STATE                    # no view yet
    ctx.set_view(np.eye(4, dtype=np.float32), 4, 4, 0.5)
    frame = torch.zeros((4, 4, 4), dtype=torch.float32, device="cuda")
    with pytest.raises(vr.VRError) as e:
        ctx.overlay_catalogue(boxes, None, None, frame, pick)  # a frame to paint but no colours
    assert e.value.status == vr.ERR_INVALID_ARG
    with pytest.raises(vr.VRError):
        ctx.overlay_pick(pick, 0, 0, 65)
