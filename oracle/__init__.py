"""oracle -- TEST INFRASTRUCTURE: ctypes face of oracle/vr_oracle.c (double-precision CPU
statement of the bricked ray-casting path of arXiv:1205.0282; citations in the C header).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may
import this package. It never imports paper_1205_0282_b200 and shares no code with it.
"""
import ctypes
import os

import numpy as np

from . import build as _build

ALPHA, MIP = 0, 1
FLAG_ERT_MARGIN, FLAG_OWNER_MARGIN, FLAG_LAST_SAMPLE, FLAG_GRAZING, FLAG_NAN_MARGIN = 1, 2, 4, 8, 16

_lib = None


def lib():
    global _lib
    if _lib is None:
        L = ctypes.CDLL(_build.build())
        vp, i64, ci, dbl = ctypes.c_void_p, ctypes.c_int64, ctypes.c_int, ctypes.c_double
        L.vro_create.restype = vp
        L.vro_create.argtypes = [i64, i64, i64, ci, ci]
        L.vro_set_dense.argtypes = [vp, vp]
        L.vro_set_procedural.argtypes = [vp, vp, vp]
        L.vro_destroy.argtypes = [vp]
        L.vro_num_bricks.argtypes = [vp]
        L.vro_ghost_violations.restype = i64
        L.vro_ghost_violations.argtypes = [vp]
        L.vro_brick_data.restype = vp
        L.vro_brick_data.argtypes = [vp, ci, vp]
        L.vro_set_tf.argtypes = [vp, vp, ci, dbl, dbl]
        L.vro_brick_minmax.argtypes = [vp, ci, vp, vp]
        L.vro_brick_transparent.argtypes = [vp, ci]
        L.vro_set_tau.argtypes = [vp, dbl]
        L.vro_set_nan_limit_scale.argtypes = [vp, dbl]
        L.vro_set_ert_margin.argtypes = [vp, dbl]
        L.vro_set_order_override.argtypes = [vp, vp]
        L.vro_brick_order.argtypes = [vp, vp, vp, vp]
        L.vro_rects.argtypes = [vp, vp, vp, ci, ci, vp]
        L.vro_render.argtypes = [vp, vp, vp, ci, ci, dbl, ci, vp, i64, vp, vp, vp, vp, ci]
        L.vro_ray_bricks.argtypes = [vp, vp, vp, ci, ci, vp, i64, vp, vp, ci, vp]
        L.vro_composite.argtypes = [vp, vp, vp, ci, ci, ci, vp, i64, vp, ci]
        _lib = L
    return _lib


def _threads(n):
    if n:
        return int(n)
    try:
        return max(1, len(os.sched_getaffinity(0)))
    except AttributeError:
        return max(1, os.cpu_count() or 1)


def _f32(m):
    a = np.ascontiguousarray(np.asarray(m, dtype=np.float32).reshape(16))
    return a


class Volume:
    """Oracle volume: dense float32 [nz][ny][nx] array, or procedural (voxel function pointer)."""

    def __init__(self, nx, ny, nz, brick, ghost=1, data=None, voxel_fn=None):
        self.nx, self.ny, self.nz, self.brick, self.ghost = int(nx), int(ny), int(nz), int(brick), int(ghost)
        self._h = lib().vro_create(self.nx, self.ny, self.nz, self.brick, self.ghost)
        if not self._h:
            raise ValueError("bad volume parameters")
        self._keep = None
        if data is not None:
            d = np.ascontiguousarray(data, dtype=np.float32)
            assert d.shape == (self.nz, self.ny, self.nx)
            if lib().vro_set_dense(self._h, d.ctypes.data) != 0:
                raise MemoryError("oracle brick build failed")
        elif voxel_fn is not None:
            fn, ctx = voxel_fn
            self._keep = voxel_fn
            lib().vro_set_procedural(self._h, fn, ctx)
        self.nbricks = lib().vro_num_bricks(self._h)
        self.tau = 0.99
        self.ert_margin = 1e-5

    def __del__(self):
        try:
            if self._h:
                lib().vro_destroy(self._h)
        except Exception:
            pass

    def set_transfer_function(self, rgba, vmin, vmax):
        t = np.ascontiguousarray(rgba, dtype=np.float32)
        assert t.ndim == 2 and t.shape[1] == 4
        if lib().vro_set_tf(self._h, t.ctypes.data, t.shape[0], float(vmin), float(vmax)) != 0:
            raise ValueError("bad transfer function")

    def set_early_termination(self, tau):
        self.tau = float(tau)
        lib().vro_set_tau(self._h, self.tau)

    def set_ert_margin(self, margin):
        """R12 test hook: a termination test with |A_b - tau| < margin flags its pixel (default 1e-5)."""
        self.ert_margin = float(margin)
        lib().vro_set_ert_margin(self._h, self.ert_margin)

    def set_nan_limit_scale(self, scale):
        """R12/R14 test hook: R14's drop limit times `scale` (1 = nominal)."""
        lib().vro_set_nan_limit_scale(self._h, float(scale))

    def set_order_override(self, order):
        if order is None:
            lib().vro_set_order_override(self._h, None)
        else:
            o = np.ascontiguousarray(order, dtype=np.int32)
            assert o.size == self.nbricks
            lib().vro_set_order_override(self._h, o.ctypes.data)

    def ghost_violations(self):
        return int(lib().vro_ghost_violations(self._h))

    def brick_data(self, b):
        dims = (ctypes.c_int64 * 3)()
        p = lib().vro_brick_data(self._h, int(b), dims)
        d0, d1, d2 = dims[0], dims[1], dims[2]
        buf = (ctypes.c_float * (d0 * d1 * d2)).from_address(p)
        return np.frombuffer(buf, dtype=np.float32).reshape(d2, d1, d0).copy()

    def brick_minmax(self, b=-1):
        """(min, max) as float32 over brick b's ghost-padded cells; b = -1: the whole volume (row f1)."""
        mn, mx = ctypes.c_float(), ctypes.c_float()
        if lib().vro_brick_minmax(self._h, int(b), ctypes.byref(mn), ctypes.byref(mx)) != 0:
            raise ValueError("no data")
        return np.float32(mn.value), np.float32(mx.value)

    def brick_transparent(self, b):
        """R16: True iff the current transfer function is zero-alpha over everything brick b can sample."""
        r = lib().vro_brick_transparent(self._h, int(b))
        if r < 0:
            raise ValueError("no data or no transfer function")
        return bool(r)

    def brick_order(self, view, proj):
        o = np.empty(self.nbricks, dtype=np.int32)
        v, p = _f32(view), _f32(proj)
        if lib().vro_brick_order(self._h, v.ctypes.data, p.ctypes.data, o.ctypes.data) != 0:
            raise ValueError("singular view")
        return o

    def rects(self, view, proj, width, height):
        r = np.empty((self.nbricks, 4), dtype=np.int32)
        v, p = _f32(view), _f32(proj)
        if lib().vro_rects(self._h, v.ctypes.data, p.ctypes.data, int(width), int(height), r.ctypes.data) != 0:
            raise ValueError("singular view")
        return r

    def render(self, view, proj, width, height, step, mode, pixels=None, want_sub=False, nthreads=None):
        """Returns dict(image, flags, counts[, sub]). Full frame: image [H][W][4] float64
        (row 0 = bottom); pixel list [(i,j)...]: image [npix][4]."""
        v, p = _f32(view), _f32(proj)
        if pixels is None:
            n, pp, pix = int(width) * int(height), None, None
        else:
            pix = np.ascontiguousarray(pixels, dtype=np.int32).reshape(-1, 2)
            n, pp = pix.shape[0], pix.ctypes.data
        out = np.empty((n, 4), dtype=np.float64)
        flags = np.empty(n, dtype=np.uint8)
        counts = np.empty((n, 2), dtype=np.int64)
        sub = np.empty((n, self.nbricks, 4), dtype=np.float64) if want_sub else None
        rc = lib().vro_render(self._h, v.ctypes.data, p.ctypes.data, int(width), int(height), float(step), int(mode),
                              pp, n, out.ctypes.data, flags.ctypes.data, counts.ctypes.data,
                              sub.ctypes.data if want_sub else None, _threads(nthreads))
        if rc != 0:
            raise ValueError("vro_render failed (%d)" % rc)
        if pixels is None:
            out = out.reshape(height, width, 4)
            flags = flags.reshape(height, width)
            counts = counts.reshape(height, width, 2)
        res = dict(image=out, flags=flags, counts=counts, ert_margin=self.ert_margin)
        if want_sub:
            res["sub"] = sub

        def alt(dtau=0.0, nan_scale=1.0):
            """R12: the same frame with every marginal decision taken the other way - early termination tested
            against tau + dtau (|dtau| = the 1e-5 flag margin), R14's drop limit scaled by nan_scale (0.5 or 2,
            the flag's band). A flagged pixel has more than one correct value; these are the others."""
            tau0 = self.tau
            try:
                self.set_early_termination(tau0 + dtau)
                self.set_nan_limit_scale(nan_scale)
                return self.render(view, proj, width, height, step, mode, pixels=pixels, want_sub=want_sub, nthreads=nthreads)
            finally:
                self.set_early_termination(tau0)
                self.set_nan_limit_scale(1.0)

        res["alt"] = alt
        return res

    def ray_bricks(self, view, proj, width, height, pixels, maxlen=64):
        v, p = _f32(view), _f32(proj)
        pix = np.ascontiguousarray(pixels, dtype=np.int32).reshape(-1, 2)
        n = pix.shape[0]
        counts = np.zeros(n, dtype=np.int32)
        lists = np.full((n, maxlen), -1, dtype=np.int32)
        graz = np.zeros(n, dtype=np.uint8)
        rc = lib().vro_ray_bricks(self._h, v.ctypes.data, p.ctypes.data, int(width), int(height), pix.ctypes.data, n,
                                  counts.ctypes.data, lists.ctypes.data, int(maxlen), graz.ctypes.data)
        if rc != 0:
            raise ValueError("vro_ray_bricks failed (%d)" % rc)
        return counts, lists, graz


def composite(layers, rects, order, width, height, pixels=None, nthreads=None):
    """Front-to-back `over` of premultiplied RGBA float32 sub-images (double arithmetic)."""
    n = len(layers)
    keep = [np.ascontiguousarray(l, dtype=np.float32) for l in layers]
    ptrs = (ctypes.c_void_p * n)(*[k.ctypes.data for k in keep])
    r = np.ascontiguousarray(rects, dtype=np.int32).reshape(n, 4)
    o = np.ascontiguousarray(order, dtype=np.int32)
    if pixels is None:
        npix, pp = width * height, None
    else:
        pix = np.ascontiguousarray(pixels, dtype=np.int32).reshape(-1, 2)
        npix, pp = pix.shape[0], pix.ctypes.data
    out = np.empty((npix, 4), dtype=np.float64)
    lib().vro_composite(ptrs, r.ctypes.data, o.ctypes.data, n, int(width), int(height), pp, npix, out.ctypes.data, _threads(nthreads))
    return out.reshape(height, width, 4) if pixels is None else out
