"""Thin Python binding of libvr (include/vr.h): argument marshalling only.

Every step of the path runs in the CUDA kernels of paper_1012_2909_b200/csrc; PyTorch supplies device
memory (tensors) and the stream.  There is no CPU fallback: importing this module without the
built library, or calling it without a CUDA device, fails loudly.  It never touches oracle/.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libvr.so")

OK, ERR_INVALID_ARG, ERR_BUFFER, ERR_CUDA, ERR_STATE, ERR_UNSUPPORTED = 0, -1, -2, -3, -4, -5
MODE_MIP, MODE_EA = 0, 1
OPT_SKIP, OPT_VARIANT, OPT_CELL_SKIP, OPT_L2_FETCH, OPT_LAYOUT, OPT_DENSE, OPT_OCCUPANCY, OPT_RING, OPT_VOXEL_TYPE, OPT_MIP_TILES = 1, 2, 3, 4, 5, 6, 7, 8, 9, 10
VOXEL_F32, VOXEL_F16 = 0, 1
STATIC_MAX_PARTIALS = 4096          # VR_STATIC_MAX_PARTIALS: partial images vr_composite_bricks_static folds per call

EXPORTS = [
    "vr_create", "vr_destroy", "vr_last_error", "vr_status_string", "vr_cube_layout",
    "vr_upload_cube", "vr_generate_cube", "vr_attach_cube", "vr_download_brick", "vr_set_view",
    "vr_set_viewport", "vr_set_transfer_function", "vr_render_mip", "vr_render_ea",
    "vr_sort_bricks", "vr_partial_layout", "vr_render_bricks", "vr_composite_bricks",
    "vr_get_counters", "vr_reset_counters", "vr_set_option", "vr_get_plan",
    "vr_set_brick_window", "vr_window_layout", "vr_sort_groups", "vr_overlay_catalogue", "vr_overlay_pick", "vr_pyramid_layout", "vr_build_pyramid",
    "vr_touch_layout", "vr_measure_touch", "vr_touch_count", "vr_fold_peers", "vr_ipc_export", "vr_ipc_open",
    "vr_cube_layout_typed", "vr_render_sortlast", "vr_meta_static_bytes", "vr_composite_bricks_static",
]


class VRError(RuntimeError):
    def __init__(self, status, text):
        super().__init__(f"libvr: {text} (status {status})")
        self.status = status


class GenParams(C.Structure):
    _fields_ = [("h_sources", C.POINTER(C.c_double)), ("n_sources", C.c_int),
                ("h_zero_boxes", C.POINTER(C.c_int)), ("n_zero_boxes", C.c_int),
                ("continuum", C.c_double)]


class Partial(C.Structure):
    _fields_ = [("brick", C.c_int), ("x0", C.c_int), ("y0", C.c_int), ("w", C.c_int), ("h", C.c_int),
                ("d_data", C.c_void_p), ("pitch_px", C.c_size_t)]


class Catalogue(C.Structure):
    _fields_ = [("d_boxes", C.c_void_p), ("d_colours", C.c_void_p), ("d_visible", C.c_void_p), ("n", C.c_int)]


class PyramidLevel(C.Structure):
    _fields_ = [("width", C.c_int), ("height", C.c_int), ("tiles_x", C.c_int), ("tiles_y", C.c_int), ("offset", C.c_size_t)]


class Counters(C.Structure):
    _fields_ = [("rays", C.c_int64), ("nominal_samples", C.c_int64), ("taken_samples", C.c_int64),
                ("bricks_visited", C.c_int64), ("bricks_skipped", C.c_int64),
                ("rays_terminated", C.c_int64), ("kernel_launches", C.c_int64)]


_lib = None


def load():
    """Load libvr.so (built in-tree by paper_1012_2909_b200/build.py).  Raises if it is missing."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} is missing: run `python -m paper_1012_2909_b200.build` "
                          "(__graft_entry__.build()).  There is no CPU fallback.")
    lib = C.CDLL(LIB_PATH)
    vp, ip, fp, sz = C.c_void_p, C.POINTER(C.c_int), C.POINTER(C.c_float), C.c_size_t
    lib.vr_create.argtypes = [C.POINTER(vp), C.c_int]
    lib.vr_destroy.argtypes = [vp]
    lib.vr_last_error.argtypes = [vp]; lib.vr_last_error.restype = C.c_char_p
    lib.vr_status_string.argtypes = [C.c_int]; lib.vr_status_string.restype = C.c_char_p
    lib.vr_cube_layout.argtypes = [C.c_int] * 6 + [C.POINTER(sz), C.POINTER(sz)]
    lib.vr_upload_cube.argtypes = [vp, vp, C.c_int] + [C.c_int] * 6 + [vp, vp, vp]
    lib.vr_generate_cube.argtypes = [vp, C.POINTER(GenParams), C.c_uint64] + [C.c_int] * 6 + [vp, vp, vp]
    lib.vr_attach_cube.argtypes = [vp] + [C.c_int] * 6 + [vp, vp]
    lib.vr_download_brick.argtypes = [vp, C.c_int, vp, vp]
    lib.vr_set_view.argtypes = [vp, fp, C.c_int, C.c_int, C.c_float]
    lib.vr_set_viewport.argtypes = [vp, C.c_int, C.c_int, sz]
    lib.vr_set_transfer_function.argtypes = [vp, fp, C.c_float, C.c_float]
    lib.vr_render_mip.argtypes = [vp, vp, vp, C.c_float, vp]
    lib.vr_render_ea.argtypes = [vp, vp, fp, C.c_float, vp]
    lib.vr_sort_bricks.argtypes = [vp, C.c_int, ip, ip]
    lib.vr_partial_layout.argtypes = [vp, C.c_int, ip, C.c_int, C.POINTER(Partial), C.POINTER(sz)]
    lib.vr_render_bricks.argtypes = [vp, C.c_int, C.POINTER(Partial), C.c_int, C.c_float, vp]
    lib.vr_composite_bricks.argtypes = [vp, C.c_int, C.POINTER(Partial), C.c_int, vp, fp, vp]
    lib.vr_composite_bricks_static.argtypes = [vp, C.c_int, C.POINTER(Partial), C.c_int, vp, fp, vp]
    lib.vr_get_counters.argtypes = [vp, C.POINTER(Counters), vp]
    lib.vr_reset_counters.argtypes = [vp, vp]
    lib.vr_set_option.argtypes = [vp, C.c_int, C.c_int]
    lib.vr_get_plan.argtypes = [vp, C.c_int, C.POINTER(C.c_int), vp]
    lib.vr_set_brick_window.argtypes = [vp, C.c_int, C.c_int]
    lib.vr_window_layout.argtypes = [C.c_int] * 8 + [C.POINTER(sz), C.POINTER(sz)]
    lib.vr_sort_groups.argtypes = [vp, ip, C.c_int, ip]
    lib.vr_overlay_catalogue.argtypes = [vp, C.POINTER(Catalogue), vp, vp, vp]
    lib.vr_overlay_pick.argtypes = [vp, vp, C.c_int, C.c_int, C.c_int, ip, vp]
    lib.vr_pyramid_layout.argtypes = [C.c_int, C.c_int, C.c_int, ip, C.POINTER(PyramidLevel), C.POINTER(sz)]
    lib.vr_build_pyramid.argtypes = [vp, vp, C.c_int, C.c_int, sz, C.c_int, vp, vp]
    lib.vr_touch_layout.argtypes = [vp, C.POINTER(sz)]
    lib.vr_measure_touch.argtypes = [vp, C.c_int, C.POINTER(Partial), C.c_int, C.c_float, vp, C.c_int, vp]
    lib.vr_touch_count.argtypes = [vp, vp, C.POINTER(C.c_uint64), vp]
    lib.vr_render_sortlast.argtypes = [vp, C.c_int, C.c_float, vp, sz, C.POINTER(sz), vp, fp, vp]
    lib.vr_cube_layout_typed.argtypes = [C.c_int] * 9 + [C.POINTER(sz), C.POINTER(sz)]
    lib.vr_meta_static_bytes.argtypes = [C.c_int] * 9 + [C.POINTER(sz)]
    lib.vr_fold_peers.argtypes = [vp, C.c_int, C.POINTER(vp), ip, C.c_int, C.c_int, C.c_int, sz, C.c_int, C.c_int,
                                  C.POINTER(vp), C.c_int, sz, fp, vp]
    lib.vr_ipc_export.argtypes = [vp, vp, C.c_char_p, C.POINTER(sz)]
    lib.vr_ipc_open.argtypes = [vp, C.c_char_p, sz, C.POINTER(vp)]
    _lib = lib
    return lib


def _stream(stream):
    if stream is not None:
        return C.c_void_p(int(stream))
    import torch
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


def _f32(a, n):
    a = np.ascontiguousarray(a, dtype=np.float32).reshape(-1)
    if a.size != n:
        raise ValueError(f"expected {n} floats, got {a.size}")
    return a


def cube_layout(dims, brick):
    cb, mb = C.c_size_t(0), C.c_size_t(0)
    rc = load().vr_cube_layout(*(int(v) for v in dims), *(int(v) for v in brick), C.byref(cb), C.byref(mb))
    if rc != OK:
        raise VRError(rc, "vr_cube_layout: invalid argument")
    return cb.value, mb.value


def cube_layout_typed(dims, brick, voxel_type=VOXEL_F32, first_brick=0, end_brick=-1):
    """Bytes of the cube and meta buffers for the micro-block layout with a stored voxel type (and a brick window)."""
    cb, mb = C.c_size_t(0), C.c_size_t(0)
    rc = load().vr_cube_layout_typed(*(int(v) for v in dims), *(int(v) for v in brick), int(voxel_type), int(first_brick),
                                     int(end_brick), C.byref(cb), C.byref(mb))
    if rc != OK:
        raise VRError(rc, "vr_cube_layout_typed: invalid argument")
    return cb.value, mb.value


def meta_static_bytes(dims, brick, voxel_type=VOXEL_F32, first_brick=0, end_brick=-1):
    """Leading bytes of the meta buffer that depend on the cube alone (vr_meta_static_bytes)."""
    nb = C.c_size_t(0)
    rc = load().vr_meta_static_bytes(*(int(v) for v in dims), *(int(v) for v in brick), int(voxel_type), int(first_brick),
                                     int(end_brick), C.byref(nb))
    if rc != OK:
        raise VRError(rc, "vr_meta_static_bytes: invalid argument")
    return nb.value


def window_layout(dims, brick, first_brick, end_brick):
    cb, mb = C.c_size_t(0), C.c_size_t(0)
    rc = load().vr_window_layout(*(int(v) for v in dims), *(int(v) for v in brick), int(first_brick), int(end_brick),
                                 C.byref(cb), C.byref(mb))
    if rc != OK:
        raise VRError(rc, "vr_window_layout: invalid argument")
    return cb.value, mb.value


def pyramid_layout(width, height, tile=256):
    """[(width, height, tiles_x, tiles_y, offset), ...] and the bytes of the whole pyramid buffer."""
    lv = (PyramidLevel * 32)()
    n, nbytes = C.c_int(0), C.c_size_t(0)
    rc = load().vr_pyramid_layout(int(width), int(height), int(tile), C.byref(n), lv, C.byref(nbytes))
    if rc != OK:
        raise VRError(rc, "vr_pyramid_layout: invalid argument")
    return [(lv[i].width, lv[i].height, lv[i].tiles_x, lv[i].tiles_y, lv[i].offset) for i in range(n.value)], nbytes.value


class Context:
    """One vr_ctx.  Methods are the C calls of include/vr.h, same names minus the `vr_` prefix."""

    def __init__(self, device: int = 0):
        self._lib = load()
        self._h = C.c_void_p(None)
        rc = self._lib.vr_create(C.byref(self._h), int(device))
        if rc != OK:
            raise VRError(rc, "vr_create failed (no CUDA device? there is no CPU fallback)")
        self.dims = self.brick = None

    def close(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            self._lib.vr_destroy(self._h)
            self._h = C.c_void_p(None)

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check(self, rc):
        if rc != OK:
            raise VRError(rc, self._lib.vr_last_error(self._h).decode() or
                          self._lib.vr_status_string(rc).decode())

    # ---- S0
    def upload_cube(self, src, dims, brick, d_cube, d_meta, stream=None):
        """src: torch CUDA tensor or numpy array, float32, linear x-fastest ([nz, ny, nx])."""
        self.dims, self.brick = tuple(int(v) for v in dims), tuple(int(v) for v in brick)
        if isinstance(src, np.ndarray):
            src = np.ascontiguousarray(src, dtype=np.float32)
            ptr, on_dev = src.ctypes.data, 0
        else:
            assert src.is_cuda and src.is_contiguous() and src.dtype.is_floating_point and src.element_size() == 4
            ptr, on_dev = src.data_ptr(), 1
        self._check(self._lib.vr_upload_cube(self._h, C.c_void_p(ptr), on_dev, *self.dims, *self.brick,
                                             C.c_void_p(d_cube.data_ptr()), C.c_void_p(d_meta.data_ptr()),
                                             _stream(stream)))

    def generate_cube(self, seed, dims, brick, d_cube, d_meta, sources=None, zero_boxes=None,
                      continuum=0.0, stream=None):
        self.dims, self.brick = tuple(int(v) for v in dims), tuple(int(v) for v in brick)
        S = np.ascontiguousarray(sources if sources is not None else np.zeros((0, 16)), dtype=np.float64).reshape(-1, 16)
        Z = np.ascontiguousarray(zero_boxes if zero_boxes is not None else np.zeros((0, 6)), dtype=np.int32).reshape(-1, 6)
        p = GenParams(S.ctypes.data_as(C.POINTER(C.c_double)), S.shape[0],
                      Z.ctypes.data_as(C.POINTER(C.c_int)), Z.shape[0], float(continuum))
        self._check(self._lib.vr_generate_cube(self._h, C.byref(p), C.c_uint64(int(seed)), *self.dims, *self.brick,
                                               C.c_void_p(d_cube.data_ptr()), C.c_void_p(d_meta.data_ptr()),
                                               _stream(stream)))

    def attach_cube(self, dims, brick, d_cube, d_meta):
        self.dims, self.brick = tuple(int(v) for v in dims), tuple(int(v) for v in brick)
        self._check(self._lib.vr_attach_cube(self._h, *self.dims, *self.brick, C.c_void_p(d_cube.data_ptr()),
                                             C.c_void_p(d_meta.data_ptr())))

    def download_brick(self, brick_id, d_dst, stream=None):
        self._check(self._lib.vr_download_brick(self._h, int(brick_id), C.c_void_p(d_dst.data_ptr()), _stream(stream)))

    # ---- S1
    def set_view(self, mvp, width, height, step):
        m = _f32(mvp, 16)
        self._check(self._lib.vr_set_view(self._h, m.ctypes.data_as(C.POINTER(C.c_float)), int(width), int(height), float(step)))

    def set_viewport(self, x0, y0, pitch_px):
        self._check(self._lib.vr_set_viewport(self._h, int(x0), int(y0), int(pitch_px)))

    def set_transfer_function(self, rgba, vmin, vmax):
        t = _f32(rgba, 1024)
        self._check(self._lib.vr_set_transfer_function(self._h, t.ctypes.data_as(C.POINTER(C.c_float)), float(vmin), float(vmax)))

    # ---- S2-S4
    def render_mip(self, d_out, d_out_rgba=None, miss=0.0, stream=None):
        self._check(self._lib.vr_render_mip(self._h, C.c_void_p(d_out.data_ptr()),
                                            C.c_void_p(d_out_rgba.data_ptr()) if d_out_rgba is not None else None,
                                            float(miss), _stream(stream)))

    def render_ea(self, d_out, bg=(0, 0, 0, 0), tau=0.99, stream=None):
        b = (C.c_float * 4)(*[float(x) for x in bg])
        self._check(self._lib.vr_render_ea(self._h, C.c_void_p(d_out.data_ptr()), b, float(tau), _stream(stream)))

    # ---- S5
    def sort_bricks(self, mode):
        g = [-(-n // min(b, n)) for n, b in zip(self.dims, self.brick)]
        order = np.zeros(g[0] * g[1] * g[2], dtype=np.int32)
        n = C.c_int(0)
        self._check(self._lib.vr_sort_bricks(self._h, int(mode), order.ctypes.data_as(C.POINTER(C.c_int)), C.byref(n)))
        return order[:n.value].copy()

    def partial_layout(self, mode, brick_ids):
        ids = np.ascontiguousarray(brick_ids, dtype=np.int32)
        parts = (Partial * max(1, ids.size))()
        nbytes = C.c_size_t(0)
        self._check(self._lib.vr_partial_layout(self._h, int(mode), ids.ctypes.data_as(C.POINTER(C.c_int)), int(ids.size),
                                                parts, C.byref(nbytes)))
        return parts, int(ids.size), nbytes.value

    @staticmethod
    def bind_partials(parts, n, d_arena):
        """Turn the arena offsets written by partial_layout into device pointers."""
        base = d_arena.data_ptr()
        for i in range(n):
            parts[i].d_data = base + (parts[i].d_data or 0)
        return parts

    def render_bricks(self, mode, parts, n, tau=0.99, stream=None):
        self._check(self._lib.vr_render_bricks(self._h, int(mode), parts, int(n), float(tau), _stream(stream)))

    def composite_bricks(self, mode, parts, n, d_out, bg=(0, 0, 0, 0), stream=None):
        b = (C.c_float * 4)(*[float(x) for x in bg])
        self._check(self._lib.vr_composite_bricks(self._h, int(mode), parts, int(n), C.c_void_p(d_out.data_ptr()), b, _stream(stream)))

    def composite_bricks_static(self, mode, parts, n, d_out, bg=(0, 0, 0, 0), stream=None):
        """vr_composite_bricks without any allocation: descriptors in the library's static device array (n <= STATIC_MAX_PARTIALS)."""
        b = (C.c_float * 4)(*[float(x) for x in bg])
        self._check(self._lib.vr_composite_bricks_static(self._h, int(mode), parts, int(n), C.c_void_p(d_out.data_ptr()), b, _stream(stream)))

    def render_sortlast(self, mode, d_arena, d_out, bg=(0, 0, 0, 0), tau=0.99, stream=None):
        """One sort-last frame / panel in one call.  Returns (ok, needed_bytes): ok is False if d_arena (a uint8 CUDA tensor
        or None) is smaller than needed_bytes and nothing was rendered."""
        b = (C.c_float * 4)(*[float(x) for x in bg])
        need = C.c_size_t(0)
        ptr = C.c_void_p(d_arena.data_ptr()) if d_arena is not None else None
        rc = self._lib.vr_render_sortlast(self._h, int(mode), float(tau), ptr, int(d_arena.numel()) if d_arena is not None else 0,
                                          C.byref(need), C.c_void_p(d_out.data_ptr()), b, _stream(stream))
        if rc == ERR_BUFFER:
            return False, need.value
        self._check(rc)
        return True, need.value

    # ---- sharded sort-last: exchange + fold + gather in one kernel over peer memory
    def fold_peers(self, mode, frame_ptrs, order, width, height, pitch_px, y0, rows, out_ptrs, out_pitch_px, bg=(0, 0, 0, 0),
                   stream=None):
        """frame_ptrs / out_ptrs: device addresses (ints) of every rank's partial frame / final frame."""
        n, n_out = len(frame_ptrs), len(out_ptrs)
        fin = (C.c_void_p * n)(*[int(p) for p in frame_ptrs])
        fout = (C.c_void_p * n_out)(*[int(p) for p in out_ptrs])
        order = np.ascontiguousarray(order, dtype=np.int32)
        b = (C.c_float * 4)(*[float(x) for x in bg])
        self._check(self._lib.vr_fold_peers(self._h, int(mode), fin, order.ctypes.data_as(C.POINTER(C.c_int)), n, int(width),
                                            int(height), int(pitch_px), int(y0), int(rows), fout, n_out, int(out_pitch_px), b,
                                            _stream(stream)))

    def ipc_export(self, tensor):
        """(handle bytes, offset) naming a CUDA tensor's memory for another process (CUDA IPC)."""
        h = C.create_string_buffer(64)
        off = C.c_size_t(0)
        self._check(self._lib.vr_ipc_export(self._h, C.c_void_p(tensor.data_ptr()), h, C.byref(off)))
        return h.raw, off.value

    def ipc_open(self, handle, offset):
        """Device address in THIS process of memory exported by a peer process."""
        p = C.c_void_p(None)
        self._check(self._lib.vr_ipc_open(self._h, C.c_char_p(handle), int(offset), C.byref(p)))
        return p.value

    # ---- B_touch measurement
    def touch_layout(self):
        n = C.c_size_t(0)
        self._check(self._lib.vr_touch_layout(self._h, C.byref(n)))
        return n.value

    def measure_touch(self, mode, parts, n, d_bitmap, tau=0.99, accumulate=False, stream=None):
        self._check(self._lib.vr_measure_touch(self._h, int(mode), parts, int(n), float(tau), C.c_void_p(d_bitmap.data_ptr()),
                                               int(bool(accumulate)), _stream(stream)))

    def touch_count(self, d_bitmap, stream=None):
        out = (C.c_uint64 * 3)()
        self._check(self._lib.vr_touch_count(self._h, C.c_void_p(d_bitmap.data_ptr()), out, _stream(stream)))
        return {"sectors": int(out[0]), "lines": int(out[1]), "taken_samples": int(out[2])}

    # ---- counters / options
    def get_counters(self, stream=None):
        c = Counters()
        self._check(self._lib.vr_get_counters(self._h, C.byref(c), _stream(stream)))
        return {k: getattr(c, k) for k, _ in Counters._fields_}

    def reset_counters(self, stream=None):
        self._check(self._lib.vr_reset_counters(self._h, _stream(stream)))

    def get_plan(self, mode, stream=None):
        out = (C.c_int * 3)()
        self._check(self._lib.vr_get_plan(self._h, int(mode), out, _stream(stream)))
        return {"variant": out[0], "skip_level": out[1], "dense": out[2]}

    def set_brick_window(self, first_brick, end_brick):
        self._check(self._lib.vr_set_brick_window(self._h, int(first_brick), int(end_brick)))

    def sort_groups(self, group_first):
        g = np.ascontiguousarray(group_first, dtype=np.int32)
        order = np.zeros(g.size - 1, dtype=np.int32)
        self._check(self._lib.vr_sort_groups(self._h, g.ctypes.data_as(C.POINTER(C.c_int)), int(g.size - 1),
                                             order.ctypes.data_as(C.POINTER(C.c_int))))
        return order

    def overlay_catalogue(self, d_boxes, d_colours, d_visible, d_frame, d_pick, stream=None):
        """d_boxes: int32 CUDA tensor [n, 6]; d_colours: float32 [n, 4] or None; d_visible: uint8 [n] or None."""
        cat = Catalogue(d_boxes.data_ptr() if d_boxes is not None and d_boxes.numel() else None,
                        d_colours.data_ptr() if d_colours is not None and d_colours.numel() else None,
                        d_visible.data_ptr() if d_visible is not None else None,
                        int(d_boxes.shape[0]) if d_boxes is not None else 0)
        self._check(self._lib.vr_overlay_catalogue(self._h, C.byref(cat), C.c_void_p(d_frame.data_ptr()) if d_frame is not None else None,
                                                   C.c_void_p(d_pick.data_ptr()), _stream(stream)))

    def overlay_pick(self, d_pick, x, y, radius, stream=None):
        box = C.c_int(-1)
        self._check(self._lib.vr_overlay_pick(self._h, C.c_void_p(d_pick.data_ptr()), int(x), int(y), int(radius), C.byref(box),
                                              _stream(stream)))
        return box.value

    def build_pyramid(self, d_frame, width, height, pitch_px, d_out, tile=256, stream=None):
        self._check(self._lib.vr_build_pyramid(self._h, C.c_void_p(d_frame.data_ptr()), int(width), int(height), int(pitch_px),
                                               int(tile), C.c_void_p(d_out.data_ptr()), _stream(stream)))

    def set_option(self, option, value):
        self._check(self._lib.vr_set_option(self._h, int(option), int(value)))
