"""Pins of the reduced-precision storage definitions (oracle/oquant.py, O-16) against what the
mathematics and the IEEE formats fix: values the binary16 format prints for worked examples, the round-trip error
bounds, identity on exactly representable cubes, monotonicity (so a MIP of the quantised cube is the quantised MIP
where samples fall on voxels), and that the oracle's march of Q(cube) obeys the bound on an axis-aligned MIP."""
import numpy as np
import pytest

from oracle import oquant
from paper_1012_2909_b200 import workloads as wl


def test_f16_worked_values():
    # binary16: 10 mantissa bits; the values below are the format's own (Q(1/3) = 0x3555, spacing 2^-12 at 1/3)
    q = oquant.quantise_f16(np.array([1.0 / 3.0, 1.0, 2049.0, 2051.0, 65504.0, 6.0e-8, 2.0 ** -24, 3.0 * 2.0 ** -25, -0.1], np.float32))
    assert q[0] == np.float32(0.333251953125) and q[1] == 1.0
    assert q[2] == 2048.0 and q[3] == 2052.0                 # ties to even at spacing 2 above 2048
    assert q[4] == 65504.0
    assert q[5] == np.float32(2.0 ** -24)                    # subnormal spacing 2^-24: 6e-8 rounds to one unit
    assert q[6] == np.float32(2.0 ** -24) and q[7] == np.float32(2.0 ** -23)   # 1.5 units: tie to even = 2 units
    assert q[8] == np.float32(-0.0999755859375)
    with pytest.raises(ValueError):
        oquant.quantise_f16(np.array([70000.0], np.float32))
    with pytest.raises(ValueError):
        oquant.quantise_f16(np.array([np.nan], np.float32))


def test_f16_round_trip_bound_identity_and_monotone():
    rng = np.random.default_rng(7)
    v = (rng.normal(size=200000) * rng.choice([1e-3, 1.0, 30.0, 3000.0], size=200000)).astype(np.float32)
    q = oquant.quantise_f16(v)
    big = np.abs(v) >= 2.0 ** -14
    assert (np.abs(q[big].astype(np.float64) - v[big]) <= 2.0 ** -11 * np.abs(v[big].astype(np.float64))).all()
    assert (np.abs(q[~big].astype(np.float64) - v[~big]) <= 2.0 ** -25).all()
    assert np.array_equal(oquant.quantise_f16(q), q)                                  # idempotent
    ints = np.arange(-2048, 2049, dtype=np.float32)
    assert np.array_equal(oquant.quantise_f16(ints), ints)                            # exactly representable: identity
    order = np.argsort(v, kind="stable")
    assert (np.diff(q[order]) >= 0).all()                                             # monotone


def test_u8_per_brick_round_trip_bound_and_identity():
    rng = np.random.default_rng(9)
    cube = rng.normal(size=(20, 33, 41)).astype(np.float32) * 3.0
    bricks = oquant.quantise_u8_bricks(cube, (16, 16, 16))
    assert len(bricks) == 3 * 3 * 2
    for bid, (lo, scale, deq) in bricks.items():
        b = (bid % 3, (bid // 3) % 3, bid // 9)
        o = (16 * b[0], 16 * b[1], 16 * b[2])
        reg = cube[o[2]:min(o[2] + 16, 19) + 1, o[1]:min(o[1] + 16, 32) + 1, o[0]:min(o[0] + 16, 40) + 1]
        assert deq.shape == reg.shape
        assert np.abs(deq.astype(np.float64) - reg).max() <= scale / 2 + 1e-6
        assert abs(lo - reg.min()) < 1e-12 and abs(lo + 255 * scale - reg.max()) < 1e-9
    # a brick whose values are lo + k * scale exactly is reproduced exactly; a constant brick too
    exact = (np.arange(256, dtype=np.float64).reshape(4, 8, 8) * 0.125 - 3.0).astype(np.float32)
    lo, scale = oquant.brick_params_u8(exact)
    code, deq = oquant.quantise_u8(exact, lo, scale)
    assert np.array_equal(deq, exact) and code.min() == 0 and code.max() == 255
    const = np.full((3, 3, 3), 2.5, np.float32)
    lo, scale = oquant.brick_params_u8(const)
    assert np.array_equal(oquant.quantise_u8(const, lo, scale)[1], const)
    # monotone inside a brick
    v = np.sort(rng.normal(size=1000)).astype(np.float32)
    lo, scale = oquant.brick_params_u8(v)
    assert (np.diff(oquant.quantise_u8(v, lo, scale)[1]) >= 0).all()


def test_mip_of_the_quantised_cube_obeys_the_bound(ovr):
    """Axis-aligned MIP, rays through voxel centres: pixel = column maximum (pinned elsewhere), so on Q(cube) it is
    exactly Q(column maximum) (Q is monotone), within 2^-11 |m| of the unquantised pixel."""
    w = wl.scaled(wl.C1, "q", (24, 20, 28), (24, 20, 28), (24, 20))
    cube = ovr.generate(w.seed, w.dims, sources=wl.make_sources(w))
    qc = oquant.quantise_f16(cube)
    M, (W, H) = wl.axis_ortho_camera(w.dims, 2, +1)
    a, _, _ = ovr.render(ovr.Volume.linear(cube), M, W, H, 0.5, ovr.MIP, ovr.F32)
    b, _, _ = ovr.render(ovr.Volume.linear(qc), M, W, H, 0.5, ovr.MIP, ovr.F32)
    assert np.array_equal(b, oquant.quantise_f16(a))
    assert (np.abs(b.astype(np.float64) - a) <= 2.0 ** -11 * np.abs(a) + 1e-12).all()
