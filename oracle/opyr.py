"""oracle/opyr.py - CPU ORACLE of the output pyramid (O-15).  TEST INFRASTRUCTURE ONLY.

PAPER.md line 45 (section 3): "The rendering output is stored in TIFF format, which is converted to
the pyramidal tiled TIFF format."  The TIFF container is client-side and out of scope (DESIGN.md
section 9); what is computed here is the pixel content of such a file, as plain numpy:

  level 0   = the float RGBA frame quantised to 8 bits per channel: q = floor(clamp(c,0,1)*255 + 1/2),
              evaluated in float32 with a separately rounded product and sum;
  level l+1 = level l reduced by 2 x 2 box filtering: mean of the (up to 4) pixels of the block,
              rounded half up in integers, (sum + n/2) // n; size ceil(w/2) x ceil(h/2);
  levels go on while max(w, h) > tile; every level is cut into tile x tile tiles, row-major over
  the tiles, each tile stored contiguously (row-major, RGBA bytes), edge tiles zero padded.

Shares no code with paper_1012_2909_b200/; may be imported only by tests/.
"""
from __future__ import annotations

import numpy as np


def quantise(frame):
    f = np.asarray(frame, dtype=np.float32)
    x = np.minimum(np.maximum(f, np.float32(0.0)), np.float32(1.0))
    p = (x * np.float32(255.0)).astype(np.float32)
    return np.floor((p + np.float32(0.5)).astype(np.float32)).astype(np.uint8)


def reduce2(img):
    h, w, c = img.shape
    H2, W2 = -(-h // 2), -(-w // 2)
    out = np.zeros((H2, W2, c), dtype=np.uint8)
    for j in range(H2):                      # plain loops over blocks; rows vectorised only over x
        ys = [y for y in (2 * j, 2 * j + 1) if y < h]
        for i in range(W2):
            xs = [x for x in (2 * i, 2 * i + 1) if x < w]
            n = len(xs) * len(ys)
            s = np.zeros(c, dtype=np.int64)
            for y in ys:
                for x in xs:
                    s += img[y, x].astype(np.int64)
            out[j, i] = ((s + n // 2) // n).astype(np.uint8)
    return out


def reduce2_fast(img):
    """Same result as reduce2 for large frames (used after reduce2 == reduce2_fast was asserted)."""
    h, w, c = img.shape
    H2, W2 = -(-h // 2), -(-w // 2)
    pad = np.zeros((2 * H2, 2 * W2, c), dtype=np.int64)
    cnt = np.zeros((2 * H2, 2 * W2), dtype=np.int64)
    pad[:h, :w] = img
    cnt[:h, :w] = 1
    s = pad[0::2, 0::2] + pad[1::2, 0::2] + pad[0::2, 1::2] + pad[1::2, 1::2]
    n = cnt[0::2, 0::2] + cnt[1::2, 0::2] + cnt[0::2, 1::2] + cnt[1::2, 1::2]
    return ((s + (n // 2)[..., None]) // n[..., None]).astype(np.uint8)


def levels(frame, tile=256, fast=True):
    out = [quantise(frame)]
    while max(out[-1].shape[0], out[-1].shape[1]) > tile:
        out.append(reduce2_fast(out[-1]) if fast else reduce2(out[-1]))
    return out


def tiled(img, tile=256):
    h, w, c = img.shape
    ty, tx = -(-h // tile), -(-w // tile)
    out = np.zeros((ty * tx, tile, tile, c), dtype=np.uint8)
    for j in range(ty):
        for i in range(tx):
            blk = img[j * tile:(j + 1) * tile, i * tile:(i + 1) * tile]
            out[j * tx + i, :blk.shape[0], :blk.shape[1]] = blk
    return out


def pyramid_bytes(frame, tile=256):
    """The whole pyramid as one byte string: levels in order, each as its tiles."""
    return np.concatenate([tiled(l, tile).reshape(-1) for l in levels(frame, tile)])
