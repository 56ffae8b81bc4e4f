"""Reduced-precision cube storage for the oracle ("image cubes larger than a
single machine memory limit", line 47 the WALLABY cube).  TEST INFRASTRUCTURE ONLY, like the rest of oracle/.

Reading O-16 (the paper says nothing about storage precision beyond float32 voxels, line 57): a cube
stored with fewer bits is rendered as the cube Q(v) of its DEquantised float32 values by the unchanged method,

    frame = march(Q(cube)),   Q = dequantise o quantise,

so the oracle for a quantised cube is this module followed by oracle/ovr.  Two codes:

* float16: q = IEEE binary16 round-to-nearest-even of the float32 voxel, Q(v) = float32(q) (exact).  Single-valued
  (a voxel has one code wherever it is stored), monotone, |Q(v) - v| <= 2^-11 |v| for 2^-14 <= |v| <= 65504.
* 8 bit with a (scale, offset) pair per brick: over the brick's voxels PLUS its +1 halo layer (the set a trilinear
  footprint of the brick can touch), lo = min, hi = max, scale = (hi - lo) / 255 (1 if hi == lo), code =
  floor((v - lo) / scale + 1/2) clamped to 0..255, Q_b(v) = lo + scale * code, all in float64 and rounded once to
  float32.  The field is then defined PER BRICK (a halo voxel is coded with the parameters of the brick it is stored
  in), |Q_b(v) - v| <= scale / 2.  Defined and pinned here; the CUDA path implements float16 (VR_OPT_VOXEL_TYPE 1).
"""
from __future__ import annotations

import numpy as np


def quantise_f16(cube):
    """Q(cube) for float16 storage: float32 -> binary16 (round to nearest even) -> float32."""
    c = np.asarray(cube, dtype=np.float32)
    with np.errstate(over="ignore"):
        q = c.astype(np.float16)
    if not np.isfinite(q).all():
        raise ValueError("a voxel lies beyond the float16 range (65504) or is not finite")
    return q.astype(np.float32)


def brick_params_u8(region):
    """(lo, scale) of one brick from its halo-inclusive voxel region (float64)."""
    r = np.asarray(region, dtype=np.float64)
    lo, hi = float(r.min()), float(r.max())
    return lo, ((hi - lo) / 255.0 if hi > lo else 1.0)


def quantise_u8(region, lo, scale):
    """Q_b of a region with the brick's parameters: codes (uint8) and dequantised float32 values."""
    r = np.asarray(region, dtype=np.float64)
    code = np.clip(np.floor((r - lo) / scale + 0.5), 0, 255)
    return code.astype(np.uint8), (lo + scale * code).astype(np.float32)


def quantise_u8_bricks(cube, brick):
    """Per-brick 8-bit view of a cube [nz, ny, nx]: {brick id: (lo, scale, dequantised halo-inclusive region)}, brick
    id = bx + gx (by + gy bz), region = voxels [lo_a, min(lo_a + B_a, N_a - 1)] per axis (the +1 halo layer clipped to
    the cube)."""
    c = np.asarray(cube, dtype=np.float32)
    nz, ny, nx = c.shape
    B = [min(b, n) for b, n in zip(brick, (nx, ny, nz))]
    G = [-(-n // b) for n, b in zip((nx, ny, nz), B)]
    out = {}
    for bz in range(G[2]):
        for by in range(G[1]):
            for bx in range(G[0]):
                o = (bx * B[0], by * B[1], bz * B[2])
                reg = c[o[2]:min(o[2] + B[2], nz - 1) + 1, o[1]:min(o[1] + B[1], ny - 1) + 1, o[0]:min(o[0] + B[0], nx - 1) + 1]
                lo, scale = brick_params_u8(reg)
                out[bx + G[0] * (by + G[1] * bz)] = (lo, scale, quantise_u8(reg, lo, scale)[1])
    return out
