"""ctypes binding of the CPU oracle (oracle/ovr.cpp).  TEST INFRASTRUCTURE ONLY.

Importable only from tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs.  It shares nothing with the CUDA path; it never imports paper_1012_2909_b200's binding.
"""
from __future__ import annotations

import ctypes as C
import numpy as np

from . import build as _build

MIP, EA = 0, 1
F64, F32 = 64, 32
UNSPLIT, SPLIT_GLOBAL, SPLIT_SORTLAST = 0, 1, 2
OK, ERR_ARG, ERR_MISSING, ERR_SINGULAR = 0, -1, -2, -3


class _Volume(C.Structure):
    _fields_ = [("nx", C.c_int), ("ny", C.c_int), ("nz", C.c_int),
                ("bx", C.c_int), ("by", C.c_int), ("bz", C.c_int),
                ("bricks", C.POINTER(C.c_void_p))]


class _View(C.Structure):
    _fields_ = [("m", C.c_float * 16), ("width", C.c_int), ("height", C.c_int), ("step", C.c_float)]


class _TF(C.Structure):
    _fields_ = [("rgba", C.c_float * 1024), ("vmin", C.c_float), ("vmax", C.c_float)]


class _Params(C.Structure):
    _fields_ = [("mode", C.c_int), ("precision", C.c_int), ("split", C.c_int),
                ("pbx", C.c_int), ("pby", C.c_int), ("pbz", C.c_int),
                ("tau", C.c_float), ("bg", C.c_float * 4), ("miss", C.c_float), ("brute", C.c_int)]


class _Counters(C.Structure):
    _fields_ = [("nominal", C.c_int64), ("taken", C.c_int64), ("terminated", C.c_int64),
                ("flagged", C.c_int64)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build.build())
        _lib.ovr_noise.restype = C.c_double
        _lib.ovr_noise.argtypes = [C.c_uint64, C.c_uint64]
    return _lib


def _check(rc, what):
    if rc != OK:
        raise RuntimeError(f"oracle {what} failed: {rc}")


class Volume:
    """Cube storage for the oracle: a linear cube or a table of plain bricks."""

    def __init__(self, dims, brick, bricks):
        self.dims, self.brick = tuple(int(v) for v in dims), tuple(int(v) for v in brick)
        g = [-(-n // b) for n, b in zip(self.dims, self.brick)]
        self.grid = tuple(g)
        nb = g[0] * g[1] * g[2]
        self._keep = {}
        arr = (C.c_void_p * nb)()
        for b, a in bricks.items():
            a = np.ascontiguousarray(a, dtype=np.float32)
            self._keep[b] = a
            arr[b] = a.ctypes.data
        self._arr = arr
        self.c = _Volume(*self.dims, *self.brick, C.cast(arr, C.POINTER(C.c_void_p)))

    @classmethod
    def linear(cls, cube):
        """cube: float32 [nz, ny, nx] (x fastest)."""
        cube = np.ascontiguousarray(cube, dtype=np.float32)
        nz, ny, nx = cube.shape
        return cls((nx, ny, nz), (nx, ny, nz), {0: cube})


def _view(M, W, H, step):
    v = _View()
    v.m[:] = [float(x) for x in np.asarray(M, dtype=np.float32).reshape(16)]
    v.width, v.height, v.step = int(W), int(H), float(step)
    return v


def _tf(tf):
    if tf is None:
        return None
    table, vmin, vmax = tf
    t = _TF()
    t.rgba[:] = [float(x) for x in np.asarray(table, dtype=np.float32).reshape(1024)]
    t.vmin, t.vmax = float(vmin), float(vmax)
    return t


def _params(mode, precision, split, partition, tau, bg, miss, brute):
    p = _Params()
    p.mode, p.precision, p.split = mode, precision, split
    pb = partition if partition is not None else (0, 0, 0)
    p.pbx, p.pby, p.pbz = (int(v) for v in pb)
    p.tau, p.miss, p.brute = float(tau), float(miss), int(bool(brute))
    p.bg[:] = [float(x) for x in bg]
    return p


def render(vol, M, W, H, step, mode, precision=F64, tf=None, split=UNSPLIT, partition=None,
           tau=2.0, bg=(0, 0, 0, 0), miss=0.0, pixels=None, brute=False):
    """Returns (out, flags, counters dict).  out: [H, W, 4] / [H, W] for a full frame, or [n, 4] /
    [n] for an explicit pixel list (pixels = int array [n, 2] of (column, row))."""
    v, t = _view(M, W, H, step), _tf(tf)
    p = _params(mode, precision, split, partition, tau, bg, miss, brute)
    ch = 1 if mode == MIP else 4
    if pixels is None:
        n, pp = W * H, None
    else:
        pix = np.ascontiguousarray(pixels, dtype=np.int32).reshape(-1, 2)
        n, pp = pix.shape[0], pix.ctypes.data_as(C.POINTER(C.c_int))
    out = np.zeros((n, ch), dtype=np.float32)
    flags = np.zeros(n, dtype=np.uint8)
    cnt = _Counters()
    rc = lib().ovr_render(C.byref(vol.c), C.byref(v), C.byref(t) if t else None, C.byref(p), pp,
                          C.c_int64(n), out.ctypes.data_as(C.POINTER(C.c_float)),
                          flags.ctypes.data_as(C.POINTER(C.c_uint8)), C.byref(cnt))
    _check(rc, "render")
    counters = {k: getattr(cnt, k) for k in ("nominal", "taken", "terminated", "flagged")}
    if pixels is None:
        out = out.reshape(H, W, ch) if ch == 4 else out.reshape(H, W)
        flags = flags.reshape(H, W)
    elif ch == 1:
        out = out.reshape(n)
    return out, flags, counters


def render_brick(vol, M, W, H, step, mode, brick_id, rect, partition, precision=F64, tf=None,
                 tau=2.0, brute=False):
    v, t = _view(M, W, H, step), _tf(tf)
    p = _params(mode, precision, SPLIT_SORTLAST, partition, tau, (0, 0, 0, 0), 0.0, brute)
    x0, y0, w, h = (int(q) for q in rect)
    ch = 1 if mode == MIP else 4
    out = np.zeros((h, w, ch), dtype=np.float32)
    rc = lib().ovr_render_brick(C.byref(vol.c), C.byref(v), C.byref(t) if t else None, C.byref(p),
                                int(brick_id), x0, y0, w, h, out.ctypes.data_as(C.POINTER(C.c_float)))
    _check(rc, "render_brick")
    return out if ch == 4 else out.reshape(h, w)


def composite(mode, rects, partials, order, W, H, bg=(0, 0, 0, 0), miss=0.0, precision=F64):
    n = len(partials)
    rects = np.ascontiguousarray(rects, dtype=np.int32).reshape(n, 4)
    keep = [np.ascontiguousarray(a, dtype=np.float32) for a in partials]
    ptrs = (C.c_void_p * max(n, 1))(*[a.ctypes.data for a in keep])
    order_a = np.ascontiguousarray(order, dtype=np.int32) if order is not None else None
    ch = 1 if mode == MIP else 4
    out = np.zeros((H, W, ch), dtype=np.float32)
    bg_a = (C.c_float * 4)(*[float(x) for x in bg])
    rc = lib().ovr_composite(mode, precision, n, rects.ctypes.data_as(C.POINTER(C.c_int)),
                             C.cast(ptrs, C.POINTER(C.c_void_p)),
                             order_a.ctypes.data_as(C.POINTER(C.c_int)) if order_a is not None else None,
                             int(W), int(H), bg_a, C.c_float(miss),
                             out.ctypes.data_as(C.POINTER(C.c_float)))
    _check(rc, "composite")
    return out if ch == 4 else out.reshape(H, W)


def visibility_keys(M, W, H, step, brick, grid):
    v = _view(M, W, H, step)
    n = int(grid[0]) * int(grid[1]) * int(grid[2])
    keys = np.zeros(n, dtype=np.int32)
    persp = C.c_int(0)
    rc = lib().ovr_visibility_keys(C.byref(v), *(int(b) for b in brick), *(int(g) for g in grid),
                                   keys.ctypes.data_as(C.POINTER(C.c_int)), C.byref(persp))
    _check(rc, "visibility_keys")
    return keys, bool(persp.value)


def visibility_order(keys):
    """Front-to-back brick order: ascending key, ties by brick id (any tie order is valid, O-9)."""
    return np.argsort(keys, kind="stable").astype(np.int32)


def ray(M, W, H, step, i, j):
    v = _view(M, W, H, step)
    o, d, L = (C.c_double * 3)(), (C.c_double * 3)(), C.c_double(0)
    _check(lib().ovr_ray(C.byref(v), int(i), int(j), o, d, C.byref(L)), "ray")
    return np.array(o[:]), np.array(d[:]), L.value


def bricks_touched(M, W, H, step, dims, brick, pixels):
    v = _view(M, W, H, step)
    pix = np.ascontiguousarray(pixels, dtype=np.int32).reshape(-1, 2)
    g = [-(-n // b) for n, b in zip(dims, brick)]
    touched = np.zeros(g[0] * g[1] * g[2], dtype=np.uint8)
    rc = lib().ovr_bricks_touched(C.byref(v), *(int(n) for n in dims), *(int(b) for b in brick),
                                  pix.ctypes.data_as(C.POINTER(C.c_int)), C.c_int64(pix.shape[0]),
                                  touched.ctypes.data_as(C.POINTER(C.c_uint8)))
    _check(rc, "bricks_touched")
    return np.nonzero(touched)[0]


def bake_tf(tf, step):
    out = np.zeros((256, 4), dtype=np.float32)
    _check(lib().ovr_bake_tf(C.byref(_tf(tf)), C.c_float(step), out.ctypes.data_as(C.POINTER(C.c_float))), "bake_tf")
    return out


def tf_lookup(tf, step, v, baked=True):
    out = (C.c_double * 4)()
    _check(lib().ovr_tf_lookup(C.byref(_tf(tf)), C.c_float(step), int(baked), C.c_double(v), out), "tf_lookup")
    return np.array(out[:])


def noise(seed, idx):
    return lib().ovr_noise(C.c_uint64(seed), C.c_uint64(idx))


def generate(seed, dims, region=None, sources=None, zero_boxes=None, continuum=0.0):
    """float32 [wz, wy, wx] of the synthetic cube over region = (x0, y0, z0, wx, wy, wz)."""
    nx, ny, nz = (int(v) for v in dims)
    x0, y0, z0, wx, wy, wz = (0, 0, 0, nx, ny, nz) if region is None else (int(v) for v in region)
    out = np.zeros((wz, wy, wx), dtype=np.float32)
    S = np.ascontiguousarray(sources, dtype=np.float64).reshape(-1, 16) if sources is not None else np.zeros((0, 16))
    Z = np.ascontiguousarray(zero_boxes, dtype=np.int32).reshape(-1, 6) if zero_boxes is not None else np.zeros((0, 6), np.int32)
    rc = lib().ovr_generate(C.c_uint64(seed), nx, ny, nz, x0, y0, z0, wx, wy, wz,
                            S.ctypes.data_as(C.POINTER(C.c_double)), S.shape[0],
                            Z.ctypes.data_as(C.POINTER(C.c_int)), Z.shape[0], C.c_double(continuum),
                            out.ctypes.data_as(C.POINTER(C.c_float)))
    _check(rc, "generate")
    return out


def overlay(M, W, H, boxes, visible=None):
    """O-14 catalogue overlay: pick image [H, W] int32, 0 = no edge, else 1 + highest box id."""
    L = lib()
    B = np.ascontiguousarray(boxes, dtype=np.int32).reshape(-1, 6)
    vis = None if visible is None else np.ascontiguousarray(visible, dtype=np.uint8)
    pick = np.zeros((H, W), dtype=np.int32)
    v = _view(M, W, H, 1.0)
    _check(L.ovr_overlay(C.byref(v), B.ctypes.data_as(C.c_void_p), int(B.shape[0]),
                         vis.ctypes.data_as(C.c_void_p) if vis is not None else None,
                         pick.ctypes.data_as(C.c_void_p)), "ovr_overlay")
    return pick


def overlay_pick(pick, x, y, radius):
    L = lib()
    p = np.ascontiguousarray(pick, dtype=np.int32)
    return int(L.ovr_overlay_pick(p.ctypes.data_as(C.c_void_p), int(p.shape[1]), int(p.shape[0]), int(x), int(y), int(radius)))


def overlay_apply(frame, pick, colours):
    """Opaque wireframe: covered pixels take the colour of their box (numpy, trivial)."""
    out = np.array(frame, dtype=np.float32, copy=True)
    m = pick > 0
    out[m] = np.asarray(colours, dtype=np.float32).reshape(-1, 4)[pick[m] - 1]
    return out
