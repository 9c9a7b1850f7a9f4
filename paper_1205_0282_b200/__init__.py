"""paper_1205_0282_b200 -- thin Python binding of libvr (include/vr.h).

Argument marshalling only: every step of the path (brick store, view set-up, visibility sort,
ray casting, compositing) runs in the CUDA kernels behind the C ABI. PyTorch is used for device
memory (the caller's tensors) and streams. There is no CPU fallback: a missing library or a
missing CUDA device raises.

Names follow include/vr.h: Volume.upload / download / set_transfer_function /
set_early_termination / render / render_host, composite(), and the debug exports.
"""
import ctypes
import os

import numpy as np

ALPHA, MIP = 0, 1
SORT_LAST, FUSED = 0, 1
SAMPLER_MANUAL, SAMPLER_TEXTURE, SAMPLER_TEXTURE_HALF, SAMPLER_TEXTURE_BYTE = 0, 1, 2, 3
STEP_AUTO = 0.0  # vr_render step: the paper's per-ray step (R18)
HOST, DEVICE = 0, 1
LAYOUT_DEFAULT, LAYOUT_LINEAR, LAYOUT_TILED, LAYOUT_TILED_RELEASABLE = 0, 1, 2, 3

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libvr.so")

STATUS = {0: "VR_OK", 1: "VR_ERR_INVALID_ARG", 2: "VR_ERR_OUT_OF_MEMORY", 3: "VR_ERR_CUDA", 4: "VR_ERR_STATE"}

# every symbol include/vr.h declares (tests check the library exports each of them)
SYMBOLS = (
    "vr_volume_create", "vr_volume_create_layout", "vr_volume_destroy", "vr_volume_upload", "vr_volume_download", "vr_debug_brick_data",
    "vr_set_transfer_function", "vr_set_early_termination", "vr_volume_minmax", "vr_set_culling", "vr_set_traversal", "vr_set_sampler", "vr_volume_release_store", "vr_set_allocator", "vr_reserve_views", "vr_debug_brick_minmax", "vr_debug_tex_error", "vr_debug_tex_alpha_guard", "vr_debug_cell_flags", "vr_render", "vr_render_host", "vr_render_host_async", "vr_render_host_wait", "vr_composite", "vr_composite_static",
    "vr_num_bricks", "vr_debug_brick_order", "vr_debug_rects", "vr_debug_ray_bricks", "vr_debug_subimages",
    "vr_volume_create_part", "vr_render_part", "vr_render_part_pieces", "vr_part_rect", "vr_composite_parts", "vr_kd_partition", "vr_part_order",
    "vr_set_counting", "vr_set_timing", "vr_debug_stats", "vr_debug_stage_times", "vr_debug_probe_dram", "vr_debug_set_upload_path", "vr_launch_count", "vr_last_error",
)


class VrError(RuntimeError):
    def __init__(self, status, message):
        super().__init__("%s: %s" % (STATUS.get(status, status), message))
        self.status = status


class Stats(ctypes.Structure):
    _fields_ = [("samples", ctypes.c_int64), ("rays", ctypes.c_int64), ("work_items", ctypes.c_int64),
                ("subimage_bytes", ctypes.c_int64), ("cells_touched", ctypes.c_int64), ("sectors_touched", ctypes.c_int64),
                ("lines_touched", ctypes.c_int64),
                ("nbricks", ctypes.c_int32), ("overflow", ctypes.c_int32),
                ("ms_setup", ctypes.c_float), ("ms_raycast", ctypes.c_float), ("ms_composite", ctypes.c_float),
                ("bricks_culled", ctypes.c_int32)]


_lib = None


def lib():
    """Load libvr.so (built in-tree by paper_1205_0282_b200.build). Fails loudly if absent."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError("libvr.so is not built: run `python -m paper_1205_0282_b200.build` "
                              "(there is no CPU fallback)")
        L = ctypes.CDLL(LIB_PATH)
        vp, ci, cf, i64 = ctypes.c_void_p, ctypes.c_int, ctypes.c_float, ctypes.c_int64
        L.vr_volume_create.argtypes = [ci, ci, ci, ci, ci, ctypes.POINTER(vp)]
        L.vr_volume_create_layout.argtypes = [ci, ci, ci, ci, ci, ci, ctypes.POINTER(vp)]
        L.vr_volume_destroy.argtypes = [vp]
        L.vr_volume_destroy.restype = None
        L.vr_volume_upload.argtypes = [vp, vp, ci, ci, ci, ci, ci, ci, ci, vp]
        L.vr_volume_download.argtypes = [vp, vp, ci, ci, ci, ci, ci, ci, ci, vp]
        L.vr_debug_brick_data.argtypes = [vp, ci, vp, vp]
        L.vr_set_transfer_function.argtypes = [vp, vp, ci, cf, cf]
        L.vr_set_early_termination.argtypes = [vp, cf]
        L.vr_volume_minmax.argtypes = [vp, vp, vp, vp]
        L.vr_set_culling.argtypes = [vp, ci]
        L.vr_set_traversal.argtypes = [vp, ci]
        L.vr_set_sampler.argtypes = [vp, ci]
        L.vr_volume_release_store.argtypes = [vp, vp, vp]
        L.vr_set_allocator.argtypes = [vp, vp, vp]
        L.vr_reserve_views.argtypes = [vp, vp, vp, ci, ci, ci]
        L.vr_debug_brick_minmax.argtypes = [vp, vp]
        L.vr_debug_tex_error.argtypes = [vp, ci, ctypes.c_int64, ctypes.c_uint, vp, vp]
        L.vr_debug_tex_alpha_guard.argtypes = [vp, vp, vp, vp]
        L.vr_debug_cell_flags.argtypes = [vp, ci, vp, vp]
        L.vr_render.argtypes = [vp, vp, vp, ci, ci, cf, ci, vp, vp]
        L.vr_render_host.argtypes = [vp, vp, vp, ci, ci, cf, ci, vp, vp]
        L.vr_render_host_async.argtypes = [vp, vp, vp, ci, ci, cf, ci, vp, vp]
        L.vr_render_host_wait.argtypes = [vp]
        L.vr_composite.argtypes = [vp, vp, vp, ci, ci, ci, vp, vp]
        L.vr_composite_static.argtypes = [vp, vp, vp, ci, ci, ci, vp, vp]
        L.vr_volume_create_part.argtypes = [ci, ci, ci, ci, ci, vp, vp, ctypes.POINTER(vp)]
        L.vr_render_part.argtypes = [vp, vp, vp, ci, ci, cf, ci, vp, vp, vp]
        L.vr_part_rect.argtypes = [ci, ci, ci, ci, vp, vp, vp, vp, ci, ci, vp]
        L.vr_render_part_pieces.argtypes = [vp, vp, vp, ci, ci, cf, ci, vp, vp, ci, vp]
        L.vr_kd_partition.argtypes = [ci, ci, ci, ci, ci, vp, vp]
        L.vr_part_order.argtypes = [vp, ci, ci, vp, vp, vp]
        L.vr_composite_parts.argtypes = [vp, ci, vp, vp, vp, ci, ci, ci, vp, vp]
        L.vr_num_bricks.argtypes = [vp]
        L.vr_debug_brick_order.argtypes = [vp, vp, vp, vp]
        L.vr_debug_rects.argtypes = [vp, vp, vp, ci, ci, vp]
        L.vr_debug_ray_bricks.argtypes = [vp, vp, vp, ci, ci, vp, ci, vp, vp, ci, vp]
        L.vr_debug_subimages.argtypes = [vp, vp, ci, vp]
        L.vr_set_counting.argtypes = [vp, ci]
        L.vr_set_timing.argtypes = [vp, ci]
        L.vr_debug_stats.argtypes = [vp, ctypes.POINTER(Stats)]
        L.vr_debug_stage_times.argtypes = [vp, ci, vp]
        L.vr_debug_probe_dram.argtypes = [vp, ctypes.c_uint64, ci, ci, ci, ci, ci, ci, vp, vp, vp]
        L.vr_debug_set_upload_path.argtypes = [ci]
        L.vr_launch_count.argtypes = [vp]
        L.vr_launch_count.restype = i64
        L.vr_last_error.argtypes = [vp]
        L.vr_last_error.restype = ctypes.c_char_p
        _lib = L
    return _lib


def _require(cond, what):
    """Argument checks of the binding raise (an `assert` would vanish under python -O and let a bad pointer through)."""
    if not cond:
        raise ValueError("paper_1205_0282_b200: argument check failed: " + what)


def _mat(m):
    return np.ascontiguousarray(np.asarray(m, dtype=np.float32).reshape(16))


def _stream(stream):
    if stream is None:
        import torch
        return ctypes.c_void_p(torch.cuda.current_stream().cuda_stream)
    return ctypes.c_void_p(int(stream))


def _pixels(pixels):
    return np.ascontiguousarray(pixels, dtype=np.int32).reshape(-1, 2)


_ALLOC_KEEP = []  # the ctypes callbacks must outlive every handle created with them


def use_torch_allocator(enable=True):
    """vr_set_allocator with torch's caching allocator: handles created afterwards take their brick store, tables and
    scratch from torch.cuda.caching_allocator_alloc on the current stream and give them back with
    caching_allocator_delete, so torch sees (and can reuse) every byte the library holds. enable=False: cudaMalloc."""
    if not enable:
        if lib().vr_set_allocator(None, None, None) != 0:
            raise VrError(1, lib().vr_last_error(None).decode())
        return
    import torch

    @ctypes.CFUNCTYPE(ctypes.c_void_p, ctypes.c_size_t, ctypes.c_void_p)
    def _alloc(nbytes, _user):
        try:
            return torch.cuda.caching_allocator_alloc(int(nbytes))
        except Exception:  # torch raises on OOM: the C side wants NULL
            return None

    @ctypes.CFUNCTYPE(None, ctypes.c_void_p, ctypes.c_void_p)
    def _free(ptr, _user):
        torch.cuda.caching_allocator_delete(ptr)

    _ALLOC_KEEP.extend([_alloc, _free])
    if lib().vr_set_allocator(ctypes.cast(_alloc, ctypes.c_void_p), ctypes.cast(_free, ctypes.c_void_p), None) != 0:
        raise VrError(1, lib().vr_last_error(None).decode())


class Volume:
    """Handle of a bricked volume in HBM (vr_volume_create ... vr_volume_destroy)."""

    def __init__(self, nx, ny, nz, brick, ghost=1, layout=LAYOUT_DEFAULT, part=None):
        """part = (b0, b1): hold only the bricks b0 <= (bx,by,bz) < b1 of the grid (vr_volume_create_part)."""
        self._h = ctypes.c_void_p()
        self.nx, self.ny, self.nz, self.brick, self.ghost = int(nx), int(ny), int(nz), int(brick), int(ghost)
        self.layout = int(layout)
        self.part = None if part is None else (tuple(int(c) for c in part[0]), tuple(int(c) for c in part[1]))
        if self.part is not None:
            b0 = np.asarray(self.part[0], dtype=np.int32)
            b1 = np.asarray(self.part[1], dtype=np.int32)
            rc = lib().vr_volume_create_part(self.nx, self.ny, self.nz, self.brick, self.ghost, b0.ctypes.data, b1.ctypes.data,
                                             ctypes.byref(self._h))
        elif self.layout == LAYOUT_DEFAULT:
            rc = lib().vr_volume_create(self.nx, self.ny, self.nz, self.brick, self.ghost, ctypes.byref(self._h))
        else:
            rc = lib().vr_volume_create_layout(self.nx, self.ny, self.nz, self.brick, self.ghost, self.layout,
                                               ctypes.byref(self._h))
        if rc != 0:
            self._h = ctypes.c_void_p()
            raise VrError(rc, lib().vr_last_error(None).decode())
        self.nbricks = lib().vr_num_bricks(self._h)

    def close(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            lib().vr_volume_destroy(self._h)
            self._h = ctypes.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check(self, rc):
        if rc != 0:
            raise VrError(rc, lib().vr_last_error(self._h).decode())

    # -- brick store (a1) ---------------------------------------------------
    def _box(self, shape, origin):
        sz, sy, sx = (int(s) for s in shape)
        x0, y0, z0 = (int(o) for o in origin)
        return x0, y0, z0, sx, sy, sz

    def upload(self, data, origin=(0, 0, 0), stream=None):
        """data: float32 [sz][sy][sx] numpy array (host) or CUDA torch tensor (device)."""
        if isinstance(data, np.ndarray):
            d = np.ascontiguousarray(data, dtype=np.float32)
            _require(d.ndim == 3, 'd.ndim == 3')
            self._check(lib().vr_volume_upload(self._h, d.ctypes.data, HOST, *self._box(d.shape, origin), _stream(stream)))
        else:
            _require(data.is_cuda and data.is_contiguous() and data.dtype.is_floating_point and data.element_size() == 4, 'data.is_cuda and data.is_contiguous() and data.dtype.is_floating_point and data.element_size() == 4')
            _require(data.dim() == 3, 'data.dim() == 3')
            self._check(lib().vr_volume_upload(self._h, data.data_ptr(), DEVICE, *self._box(data.shape, origin), _stream(stream)))

    def download(self, out, origin=(0, 0, 0), stream=None):
        if isinstance(out, np.ndarray):
            _require(out.dtype == np.float32 and out.flags.c_contiguous and out.ndim == 3, 'out.dtype == np.float32 and out.flags.c_contiguous and out.ndim == 3')
            self._check(lib().vr_volume_download(self._h, out.ctypes.data, HOST, *self._box(out.shape, origin), _stream(stream)))
        else:
            _require(out.is_cuda and out.is_contiguous() and out.element_size() == 4 and out.dim() == 3, 'out.is_cuda and out.is_contiguous() and out.element_size() == 4 and out.dim() == 3')
            self._check(lib().vr_volume_download(self._h, out.data_ptr(), DEVICE, *self._box(out.shape, origin), _stream(stream)))
        return out

    def debug_brick_data(self, b):
        dims = (ctypes.c_int * 3)()
        self._check(lib().vr_debug_brick_data(self._h, int(b), None, dims))
        out = np.empty((dims[2], dims[1], dims[0]), dtype=np.float32)
        self._check(lib().vr_debug_brick_data(self._h, int(b), out.ctypes.data, dims))
        return out

    # -- classification (a6), termination (a7) --------------------------------
    def set_transfer_function(self, rgba, vmin, vmax):
        t = np.ascontiguousarray(rgba, dtype=np.float32)
        _require(t.ndim == 2 and t.shape[1] == 4, 't.ndim == 2 and t.shape[1] == 4')
        self._check(lib().vr_set_transfer_function(self._h, t.ctypes.data, t.shape[0], float(vmin), float(vmax)))

    def set_early_termination(self, tau):
        self._check(lib().vr_set_early_termination(self._h, float(tau)))

    # -- data range (f1) ---------------------------------------------------------
    def minmax(self, stream=None):
        """(min, max) of the uploaded volume as float32 (vr_volume_minmax)."""
        mn, mx = ctypes.c_float(), ctypes.c_float()
        self._check(lib().vr_volume_minmax(self._h, ctypes.byref(mn), ctypes.byref(mx), _stream(stream)))
        return np.float32(mn.value), np.float32(mx.value)

    def set_culling(self, enable):
        self._check(lib().vr_set_culling(self._h, int(bool(enable))))

    def debug_cell_flags(self, b):
        """[ncz][ncy][ncx] uint8: 1 where the 8x8x8 macro-cell of brick b is transparent under the current LUT (R19)."""
        dims = (ctypes.c_int * 3)()
        self._check(lib().vr_debug_cell_flags(self._h, int(b), None, dims))
        out = np.empty((dims[2], dims[1], dims[0]), dtype=np.uint8)
        self._check(lib().vr_debug_cell_flags(self._h, int(b), out.ctypes.data, dims))
        return out

    def set_traversal(self, traversal):
        """SORT_LAST (per-brick sub-images + compositing, the default) or FUSED (one ray through all bricks)."""
        self._check(lib().vr_set_traversal(self._h, int(traversal)))

    def set_sampler(self, sampler):
        """SAMPLER_MANUAL (hand-rolled float32 tri-linear, the default), SAMPLER_TEXTURE (3-D CUDA arrays behind texture
        objects: a second copy of the bricks; ALPHA values, exact MIP filter), SAMPLER_TEXTURE_HALF (float16 copies: the
        same at half the memory) or SAMPLER_TEXTURE_BYTE (8-bit arrays: the exact MIP filter only)."""
        self._check(lib().vr_set_sampler(self._h, int(sampler)))

    def release_store(self, stream=None):
        """vr_volume_release_store (handles created with layout=LAYOUT_TILED_RELEASABLE): the bricks become 3-D arrays one by
        one and their float32 cells go back to the device; ALPHA frames through the texture arm only afterwards. Returns
        the bytes given back."""
        freed = ctypes.c_int64()
        self._check(lib().vr_volume_release_store(self._h, ctypes.byref(freed), _stream(stream)))
        return int(freed.value)

    def debug_brick_minmax(self):
        """[nbricks][2] float32: (min, max) per brick over its ghost-padded cells."""
        mm = np.empty((self.nbricks, 2), dtype=np.float32)
        self._check(lib().vr_debug_brick_minmax(self._h, mm.ctypes.data))
        return mm

    def debug_tex_alpha_guard(self):
        """(mean macro-cell range, table slope in units of 1/n, whether ALPHA values may come from the arrays): R20's data guard."""
        rng, slope, ok = ctypes.c_float(), ctypes.c_float(), ctypes.c_int()
        self._check(lib().vr_debug_tex_alpha_guard(self._h, ctypes.byref(rng), ctypes.byref(slope), ctypes.byref(ok)))
        return float(rng.value), float(slope.value), bool(ok.value)

    def debug_tex_error(self, brick, n=1 << 20, seed=1):
        """(largest |filtered fetch - exact value| over n hashed positions of the brick, the brick's range): R23's constant."""
        err, rng = ctypes.c_float(), ctypes.c_float()
        self._check(lib().vr_debug_tex_error(self._h, int(brick), int(n), int(seed), ctypes.byref(err), ctypes.byref(rng)))
        return float(err.value), float(rng.value)

    # -- one frame (a2..a9) ---------------------------------------------------
    def render(self, view, proj, width, height, step, mode, out, stream=None):
        """out: CUDA float32 tensor [height][width][4]; asynchronous on the stream."""
        _require(out.is_cuda and out.is_contiguous() and out.element_size() == 4 and out.numel() == width * height * 4, 'out.is_cuda and out.is_contiguous() and out.element_size() == 4 and out.numel() == width * height * 4')
        v, p = _mat(view), _mat(proj)
        self._check(lib().vr_render(self._h, v.ctypes.data, p.ctypes.data, int(width), int(height), float(step), int(mode),
                                    out.data_ptr(), _stream(stream)))
        return out

    def reserve_views(self, views, projs, width, height):
        """vr_reserve_views: size the scratch for these views so that render() never allocates or synchronises."""
        v = np.ascontiguousarray(np.stack([_mat(m) for m in views]) if len(views) else np.zeros((0, 16), np.float32))
        p = np.ascontiguousarray(np.stack([_mat(m) for m in projs]) if len(projs) else np.zeros((0, 16), np.float32))
        if v.shape != p.shape:
            raise ValueError("reserve_views: as many projection as view matrices")
        self._check(lib().vr_reserve_views(self._h, v.ctypes.data, p.ctypes.data, v.shape[0], int(width), int(height)))

    def render_part(self, view, proj, width, height, step, mode, out, stream=None):
        """This handle's contribution to a sort-last frame (vr_render_part). out: CUDA float32 tensor
        [height][width][4] (ALPHA) or [height][width] (MIP: the raw maximum, -inf without a sample; a [height][width][4]
        tensor is accepted and its first width*height floats are written); returns the rectangle (x0,y0,x1,y1) outside
        which the partial frame is blank."""
        _require(out.is_cuda and out.is_contiguous() and out.element_size() == 4, "out: a contiguous float32 CUDA tensor")
        _require(out.numel() == width * height * 4 or (mode == MIP and out.numel() == width * height), "out: width*height*4 floats (MIP: or width*height)")
        v, p = _mat(view), _mat(proj)
        rect = np.zeros(4, dtype=np.int32)
        self._check(lib().vr_render_part(self._h, v.ctypes.data, p.ctypes.data, int(width), int(height), float(step), int(mode),
                                         out.data_ptr(), rect.ctypes.data, _stream(stream)))
        return tuple(int(c) for c in rect)

    def render_part_pieces(self, view, proj, width, height, step, mode, rects, pieces, stream=None):
        """vr_render_part_pieces: the handle's partial frame, composited straight into rectangle-packed pieces. rects:
        n x (x0,y0,x1,y1) inside the frame; pieces: n CUDA float32 tensors, piece q holding rects[q] as
        [y1-y0][x1-x0][4] (ALPHA) or [y1-y0][x1-x0] (MIP: raw maximum, -inf without a sample)."""
        n = len(pieces)
        r = np.ascontiguousarray(rects, dtype=np.int32).reshape(n, 4)
        per = 4 if mode == ALPHA else 1
        for t, rc_ in zip(pieces, r):
            _require(t.is_cuda and t.is_contiguous() and t.element_size() == 4, "pieces: contiguous float32 CUDA tensors")
            _require(t.numel() == (rc_[2] - rc_[0]) * (rc_[3] - rc_[1]) * per, "piece size does not match its rectangle and the mode")
        ptrs = (ctypes.c_void_p * max(n, 1))(*[t.data_ptr() for t in pieces])
        v, p = _mat(view), _mat(proj)
        self._check(lib().vr_render_part_pieces(self._h, v.ctypes.data, p.ctypes.data, int(width), int(height), float(step), int(mode),
                                                r.ctypes.data, ptrs, n, _stream(stream)))
        return pieces

    def composite_parts(self, mode, parts, rects, order, width, height, out, stream=None):
        """Merge partial frames (vr_composite_parts). parts: CUDA float32 tensors [y1-y0][x1-x0][4], piece l
        covering rects[l]; order: the pieces front to back; out: CUDA float32 tensor [height][width][4]."""
        n = len(parts)
        ptrs = (ctypes.c_void_p * max(n, 1))(*[l.data_ptr() for l in parts])
        r = np.ascontiguousarray(rects, dtype=np.int32).reshape(n, 4)
        o = np.ascontiguousarray(order, dtype=np.int32).reshape(n)
        per = 4 if mode == ALPHA else 1  # MIP pieces are scalar (one float per pixel)
        for l, rc_ in zip(parts, r):
            _require(l.is_cuda and l.is_contiguous() and l.element_size() == 4, 'l.is_cuda and l.is_contiguous() and l.element_size() == 4')
            _require(l.numel() == (rc_[2] - rc_[0]) * (rc_[3] - rc_[1]) * per, "piece size does not match its rectangle and the mode")
        _require(out.is_cuda and out.is_contiguous() and out.numel() == width * height * 4, 'out.is_cuda and out.is_contiguous() and out.numel() == width * height * 4')
        self._check(lib().vr_composite_parts(self._h, int(mode), ptrs, r.ctypes.data, o.ctypes.data, n, int(width), int(height),
                                             out.data_ptr(), _stream(stream)))
        return out

    def render_host(self, view, proj, width, height, step, mode, out=None, stream=None):
        """out: float32 numpy array or pinned CPU tensor [height][width][4]; returns when filled."""
        v, p = _mat(view), _mat(proj)
        if out is None:
            out = np.empty((height, width, 4), dtype=np.float32)
        if isinstance(out, np.ndarray):
            _require(out.dtype == np.float32 and out.flags.c_contiguous and out.size == width * height * 4, 'out.dtype == np.float32 and out.flags.c_contiguous and out.size == width * height * 4')
            ptr = out.ctypes.data
        else:
            _require((not out.is_cuda) and out.is_contiguous() and out.element_size() == 4 and out.numel() == width * height * 4, '(not out.is_cuda) and out.is_contiguous() and out.element_size() == 4 and out.numel() == width * height * 4')
            ptr = out.data_ptr()
        self._check(lib().vr_render_host(self._h, v.ctypes.data, p.ctypes.data, int(width), int(height), float(step),
                                         int(mode), ptr, _stream(stream)))
        return out

    def render_host_async(self, view, proj, width, height, step, mode, out, stream=None):
        """Pipelined render_host: `out` (pinned CPU tensor or numpy array) is filled once
        render_host_wait() has returned; use one buffer per frame in flight (two are)."""
        v, p = _mat(view), _mat(proj)
        if isinstance(out, np.ndarray):
            _require(out.dtype == np.float32 and out.flags.c_contiguous and out.size == width * height * 4, 'out.dtype == np.float32 and out.flags.c_contiguous and out.size == width * height * 4')
            ptr = out.ctypes.data
        else:
            _require((not out.is_cuda) and out.is_contiguous() and out.element_size() == 4 and out.numel() == width * height * 4, '(not out.is_cuda) and out.is_contiguous() and out.element_size() == 4 and out.numel() == width * height * 4')
            ptr = out.data_ptr()
        self._check(lib().vr_render_host_async(self._h, v.ctypes.data, p.ctypes.data, int(width), int(height), float(step),
                                               int(mode), ptr, _stream(stream)))
        return out

    def render_host_wait(self):
        self._check(lib().vr_render_host_wait(self._h))

    # -- debug / test exports ---------------------------------------------------
    def debug_brick_order(self, view, proj):
        v, p = _mat(view), _mat(proj)
        o = np.empty(self.nbricks, dtype=np.int32)
        self._check(lib().vr_debug_brick_order(self._h, v.ctypes.data, p.ctypes.data, o.ctypes.data))
        return o

    def debug_rects(self, view, proj, width, height):
        v, p = _mat(view), _mat(proj)
        r = np.empty((self.nbricks, 4), dtype=np.int32)
        self._check(lib().vr_debug_rects(self._h, v.ctypes.data, p.ctypes.data, int(width), int(height), r.ctypes.data))
        return r

    def debug_ray_bricks(self, view, proj, width, height, pixels, maxlen=64):
        v, p = _mat(view), _mat(proj)
        pix = _pixels(pixels)
        n = pix.shape[0]
        counts = np.zeros(n, dtype=np.int32)
        lists = np.full((n, maxlen), -1, dtype=np.int32)
        graz = np.zeros(n, dtype=np.uint8)
        self._check(lib().vr_debug_ray_bricks(self._h, v.ctypes.data, p.ctypes.data, int(width), int(height), pix.ctypes.data,
                                              n, counts.ctypes.data, lists.ctypes.data, int(maxlen), graz.ctypes.data))
        return counts, lists, graz

    def debug_subimages(self, pixels):
        pix = _pixels(pixels)
        out = np.empty((pix.shape[0], self.nbricks, 4), dtype=np.float32)
        self._check(lib().vr_debug_subimages(self._h, pix.ctypes.data, pix.shape[0], out.ctypes.data))
        return out

    def set_counting(self, mode):
        """0 off, 1 count samples, 2 also track the distinct cells / sectors read."""
        self._check(lib().vr_set_counting(self._h, int(mode)))

    def set_timing(self, enable):
        self._check(lib().vr_set_timing(self._h, int(bool(enable))))

    def debug_stats(self):
        s = Stats()
        self._check(lib().vr_debug_stats(self._h, ctypes.byref(s)))
        return {k: getattr(s, k) for k, _ in Stats._fields_}

    def debug_stage_times(self, nframes):
        """[nframes][3] ms of (set-up, ray cast, compositing) of the last nframes timed frames."""
        out = np.empty((int(nframes), 3), dtype=np.float32)
        self._check(lib().vr_debug_stage_times(self._h, int(nframes), out.ctypes.data))
        return out

    def launch_count(self):
        return int(lib().vr_launch_count(self._h))


def part_rect(dims, brick, box, view, proj, width, height):
    """vr_part_rect: the frame rectangle (x0,y0,x1,y1) a part's partial frame can be non-blank in. Host only."""
    b0 = np.asarray(box[0], dtype=np.int32)
    b1 = np.asarray(box[1], dtype=np.int32)
    v, p = _mat(view), _mat(proj)
    rect = np.zeros(4, dtype=np.int32)
    rc = lib().vr_part_rect(int(dims[0]), int(dims[1]), int(dims[2]), int(brick), b0.ctypes.data, b1.ctypes.data, v.ctypes.data,
                            p.ctypes.data, int(width), int(height), rect.ctypes.data)
    if rc != 0:
        raise VrError(rc, lib().vr_last_error(None).decode())
    return tuple(int(c) for c in rect)


PROBE_FLAVOURS = ("ld.global", "ld.global.nc", "ld.global.cg", "ld.global.cs", "ld.global.cv", "ld.global.nc.L1::no_allocate",
                  "ld.global.nc.L1::no_allocate.L2::64B", "ld.global.nc.L2::128B", "ld.global.nc.L2::256B", "ld.global.nc.v4",
                  "ld.global.nc.L2::64B", "tex1Dfetch.f32 (linear memory)", "tex1Dfetch.v4.f32 (linear memory)",
                  "tex3D.v4.f32 point (3-D array)", "tex3D.f32 linear (3-D array)")


def debug_probe_dram(buf, flavour, span_bytes=128, group=1, loads_per_thread=256, ctas=148 * 8, l2_fetch_granularity=0, stream=None):
    """vr_debug_probe_dram on a CUDA tensor: returns (ms of one launch, loads it issued)."""
    if not (buf.is_cuda and buf.is_contiguous()):
        raise ValueError("debug_probe_dram: buf must be a contiguous CUDA tensor")
    ms, loads = ctypes.c_float(), ctypes.c_uint64()
    rc = lib().vr_debug_probe_dram(buf.data_ptr(), buf.numel() * buf.element_size(), int(flavour), int(span_bytes), int(group),
                                   int(loads_per_thread), int(ctas), int(l2_fetch_granularity), ctypes.byref(ms), ctypes.byref(loads),
                                   _stream(stream))
    if rc != 0:
        raise VrError(rc, "vr_debug_probe_dram failed")
    return float(ms.value), int(loads.value)


def kd_partition(dims, brick, nparts):
    """vr_kd_partition: (boxes, tree) - boxes[r] = (b0, b1), the half-open box of bricks of part r;
    tree: int32 [(2 nparts - 1)][4] in libvr's encoding, for part_order. Host only."""
    nparts = int(nparts)
    boxes = np.zeros((max(nparts, 1), 6), dtype=np.int32)
    tree = np.zeros((max(2 * nparts - 1, 1), 4), dtype=np.int32)
    rc = lib().vr_kd_partition(int(dims[0]), int(dims[1]), int(dims[2]), int(brick), nparts, boxes.ctypes.data, tree.ctypes.data)
    if rc != 0:
        raise VrError(rc, lib().vr_last_error(None).decode())
    return [(tuple(int(c) for c in b[:3]), tuple(int(c) for c in b[3:])) for b in boxes], tree


def part_order(tree, brick, view, proj):
    """vr_part_order: the parts of a k-d partition front to back for this view. Host only."""
    t = np.ascontiguousarray(tree, dtype=np.int32).reshape(-1, 4)
    nparts = (t.shape[0] + 1) // 2
    v, p = _mat(view), _mat(proj)
    out = np.zeros(nparts, dtype=np.int32)
    rc = lib().vr_part_order(t.ctypes.data, nparts, int(brick), v.ctypes.data, p.ctypes.data, out.ctypes.data)
    if rc != 0:
        raise VrError(rc, lib().vr_last_error(None).decode())
    return [int(r) for r in out]


def debug_set_upload_path(path):
    """vr_debug_set_upload_path: 0 = cp.async staging (default), 1 = TMA box loads."""
    if lib().vr_debug_set_upload_path(int(path)) != 0:
        raise VrError(1, lib().vr_last_error(None).decode())


def composite(layers, rects, order, width, height, out, stream=None):
    """Stand-alone sort-last compositing (vr_composite). layers: CUDA float32 tensors
    [y1-y0][x1-x0][4] (premultiplied); rects: n x (x0,y0,x1,y1); order: front-to-back indices;
    out: CUDA float32 tensor [height][width][4]."""
    n = len(layers)
    ptrs = (ctypes.c_void_p * max(n, 1))(*[l.data_ptr() for l in layers])
    r = np.ascontiguousarray(rects, dtype=np.int32).reshape(n, 4)
    o = np.ascontiguousarray(order, dtype=np.int32).reshape(n)
    for l, rc_ in zip(layers, r):
        _require(l.is_cuda and l.is_contiguous() and l.element_size() == 4, 'l.is_cuda and l.is_contiguous() and l.element_size() == 4')
        _require(l.numel() == (rc_[2] - rc_[0]) * (rc_[3] - rc_[1]) * 4, 'l.numel() == (rc_[2] - rc_[0]) * (rc_[3] - rc_[1]) * 4')
    _require(out.is_cuda and out.is_contiguous() and out.numel() == width * height * 4, 'out.is_cuda and out.is_contiguous() and out.numel() == width * height * 4')
    rc = lib().vr_composite(ptrs, r.ctypes.data, o.ctypes.data, n, int(width), int(height), out.data_ptr(), _stream(stream))
    if rc != 0:
        raise VrError(rc, lib().vr_last_error(None).decode())
    return out


COMPOSITE_STATIC_MAX_LAYERS = 256


def composite_static(layers, rects, order, width, height, out, stream=None):
    """vr_composite_static: vr_composite without any allocation (the device tables live in a fixed array inside the
    library; at most COMPOSITE_STATIC_MAX_LAYERS layers; calls that overlap on the GPU race). Arguments as composite."""
    n = len(layers)
    ptrs = (ctypes.c_void_p * max(n, 1))(*[l.data_ptr() for l in layers])
    r = np.ascontiguousarray(rects, dtype=np.int32).reshape(n, 4)
    o = np.ascontiguousarray(order, dtype=np.int32).reshape(n)
    for l, rc_ in zip(layers, r):
        _require(l.is_cuda and l.is_contiguous() and l.element_size() == 4, 'l.is_cuda and l.is_contiguous() and l.element_size() == 4')
        _require(l.numel() == (rc_[2] - rc_[0]) * (rc_[3] - rc_[1]) * 4, 'l.numel() == (rc_[2] - rc_[0]) * (rc_[3] - rc_[1]) * 4')
    _require(out.is_cuda and out.is_contiguous() and out.numel() == width * height * 4, 'out.is_cuda and out.is_contiguous() and out.numel() == width * height * 4')
    rc = lib().vr_composite_static(ptrs, r.ctypes.data, o.ctypes.data, n, int(width), int(height), out.data_ptr(), _stream(stream))
    if rc != 0:
        raise VrError(rc, lib().vr_last_error(None).decode())
    return out
