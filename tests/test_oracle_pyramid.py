"""Pins of the output-pyramid oracle (O-15): closed forms and invariants."""
import numpy as np

from oracle import opyr


def test_quantise_table_values():
    # c = k/255 maps to k (k/255*255 + 1/2 floors to k); clamped outside [0,1]; halves round up
    k = np.arange(256)
    f = (k / 255.0).astype(np.float32).reshape(16, 16, 1).repeat(4, axis=2)
    assert np.array_equal(opyr.quantise(f)[..., 0].reshape(-1), k)
    odd = np.array([[[-0.5, 1.5, 0.001, 0.999]]], np.float32)      # 0.255 + 0.5 -> 0; 254.745 + 0.5 -> 255
    assert opyr.quantise(odd).reshape(-1).tolist() == [0, 255, 0, 255]
    assert opyr.quantise(np.full((3, 5, 4), 0.2, np.float32)).max() == 51        # 0.2 * 255 = 51


def test_reduce_closed_forms():
    const = np.full((7, 9, 4), 93, np.uint8)
    assert (opyr.reduce2(const) == 93).all() and opyr.reduce2(const).shape == (4, 5, 4)
    chk = np.zeros((8, 8, 4), np.uint8)
    chk[0::2, 1::2] = 255
    chk[1::2, 0::2] = 255                                   # every 2 x 2 block: 0 255 / 255 0 -> (510 + 2) // 4 = 128
    assert (opyr.reduce2(chk) == 128).all()
    ramp = np.arange(12, dtype=np.uint8)[None, :, None].repeat(6, 0).repeat(4, 2)   # value = x
    r = opyr.reduce2(ramp)
    assert np.array_equal(r[0, :, 0], np.array([1, 3, 5, 7, 9, 11]))             # (2x + 2x+1)*2/4 = 2x + 1/2 -> half up
    edge = np.arange(15, dtype=np.uint8).reshape(3, 5, 1).repeat(4, 2)          # odd sizes: partial blocks
    e = opyr.reduce2(edge)
    assert e.shape == (2, 3, 4)
    assert e[1, 2, 0] == 14 and e[0, 2, 0] == (4 + 9 + 1) // 2 and e[1, 0, 0] == (10 + 11 + 1) // 2


def test_fast_reduction_equals_the_plain_one():
    rng = np.random.default_rng(5)
    for shape in [(1, 1), (2, 3), (7, 5), (16, 16), (33, 18)]:
        img = rng.integers(0, 256, (*shape, 4), dtype=np.uint8)
        assert np.array_equal(opyr.reduce2(img), opyr.reduce2_fast(img))


def test_level_sizes_and_tiles_of_the_wall_frame():
    # 9600 x 5400; levels halve (rounding up) until one 256-tile holds the image
    sizes, w, h = [], 9600, 5400
    while True:
        sizes.append((w, h))
        if max(w, h) <= 256:
            break
        w, h = -(-w // 2), -(-h // 2)
    assert sizes == [(9600, 5400), (4800, 2700), (2400, 1350), (1200, 675), (600, 338), (300, 169), (150, 85)]
    small = np.zeros((85, 150, 4), np.float32)
    assert len(opyr.levels(small)) == 1 and opyr.tiled(opyr.quantise(small)).shape == (1, 256, 256, 4)
    # a pixel of a level is found in its tile at the expected place, edge tiles are zero padded
    rng = np.random.default_rng(9)
    img = rng.integers(1, 256, (300, 520, 4), dtype=np.uint8)
    t = opyr.tiled(img)
    assert t.shape == (2 * 3, 256, 256, 4)
    for (x, y) in [(0, 0), (255, 255), (256, 0), (519, 299), (300, 260)]:
        assert np.array_equal(t[(y // 256) * 3 + x // 256, y % 256, x % 256], img[y, x])
    assert not t[5, 44:, :].any() and not t[5, :, 8:].any()
    # mean brightness is preserved by the reductions up to rounding (half up: bias < 1/2 per level)
    lv = opyr.levels(rng.uniform(0, 1, (700, 900, 4)).astype(np.float32))
    assert len(lv) == 3
    for a, b in zip(lv, lv[1:]):
        assert abs(float(a.mean()) - float(b.mean())) < 0.75
