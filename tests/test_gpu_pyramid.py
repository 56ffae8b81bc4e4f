"""NEXT-3: output pyramid on the GPU against the numpy oracle (O-15; PAPER.md line
45).  Byte output: bit-exact."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def _run(torch, vr, frame_t, W, H, pitch, tile):
    levels, nbytes = vr.pyramid_layout(W, H, tile)
    out = torch.full((nbytes,), 0xAB, dtype=torch.uint8, device="cuda")
    ctx = vr.Context(0)
    ctx.build_pyramid(frame_t, W, H, pitch, out, tile)
    torch.cuda.synchronize()
    return levels, out.cpu().numpy()


@pytest.mark.parametrize("W,H,pitch,tile", [(900, 700, 900, 256), (517, 301, 640, 64), (64, 64, 64, 64), (1, 1, 1, 16),
                                            (257, 255, 300, 256)])
def test_pyramid_bytes_equal_oracle(W, H, pitch, tile):
    import torch
    from paper_1012_2909_b200 import vr
    from oracle import opyr
    g = torch.Generator(device="cuda").manual_seed(1234 + W)
    buf = torch.rand((H, pitch, 4), generator=g, device="cuda") * 1.2 - 0.1        # some values outside [0, 1]
    buf[0, 0] = torch.tensor([0.0, 1.0, 0.5, 2.0 / 255.0])
    frame = buf[:, :W].cpu().numpy()
    levels, got = _run(torch, vr, buf, W, H, pitch, tile)
    want_levels = opyr.levels(frame, tile)
    assert [(l[0], l[1]) for l in levels] == [(l.shape[1], l.shape[0]) for l in want_levels]
    assert np.array_equal(got, opyr.pyramid_bytes(frame, tile))


def test_pyramid_of_the_9600x5400_wall_frame():
    """P:37 / P:45: the tiled-display frame size; sampled tiles of every level against the oracle."""
    import torch
    from paper_1012_2909_b200 import vr
    from oracle import opyr
    W, H = 9600, 5400
    g = torch.Generator(device="cuda").manual_seed(7)
    buf = torch.rand((H, W, 4), generator=g, device="cuda")
    levels, got = _run(torch, vr, buf, W, H, W, 256)
    assert [(l[0], l[1]) for l in levels] == [(9600, 5400), (4800, 2700), (2400, 1350), (1200, 675), (600, 338), (300, 169), (150, 85)]
    want = opyr.levels(buf.cpu().numpy(), 256)
    for (w, h, tx, ty, off), img in zip(levels, want):
        tiles = got[off:off + tx * ty * 256 * 256 * 4].reshape(ty * tx, 256, 256, 4)
        ref = opyr.tiled(img, 256)
        pick = sorted({0, tx - 1, (ty - 1) * tx, ty * tx - 1, (ty // 2) * tx + tx // 2})
        for t in pick:
            assert np.array_equal(tiles[t], ref[t]), (w, h, t)
        assert int(tiles.astype(np.int64).sum()) == int(ref.astype(np.int64).sum())     # whole-level invariant


def test_pyramid_error_codes():
    import torch
    from paper_1012_2909_b200 import vr
    with pytest.raises(vr.VRError):
        vr.pyramid_layout(100, 100, 100)          # tile must be a power of two
    ctx = vr.Context(0)
    f = torch.zeros((4, 4, 4), device="cuda")
    o = torch.zeros(16 * 16 * 4, dtype=torch.uint8, device="cuda")
    with pytest.raises(vr.VRError) as e:
        ctx.build_pyramid(f, 4, 4, 2, o, 16)      # pitch < width
    assert e.value.status == vr.ERR_INVALID_ARG
