"""synth -- seeded synthetic INPUTS shared by the CPU oracle and the CUDA path.

Holds none of the method's arithmetic: it only makes cubes (noise + Gaussian sources +
optional spectral ramp), transfer-function tables, cameras (OpenGL-style matrices) and the
premultiplied layers of the compositing microbenchmark. Recipe and the datasets these stand
in for (paper Table 1): DESIGN.md "Synthetic inputs".
"""
import ctypes
import math

import numpy as np

from . import build as _build

BASE_SEED = 12050282

_cpu = None
_cuda = None


def _cpu_lib():
    global _cpu
    if _cpu is None:
        lib = ctypes.CDLL(_build.build_cpu())
        i64, u64, i32, vp, dbl = ctypes.c_int64, ctypes.c_uint64, ctypes.c_int32, ctypes.c_void_p, ctypes.c_double
        lib.vs_cube_create.restype = vp
        lib.vs_cube_create.argtypes = [u64, i64, i64, i64, i32, dbl]
        lib.vs_cube_create_kind.restype = vp
        lib.vs_cube_create_kind.argtypes = [u64, i64, i64, i64, i32, dbl, i32]
        lib.vs_cube_destroy.argtypes = [vp]
        for f in (lib.vs_cube_nprof, lib.vs_cube_ncell, lib.vs_cube_nitems):
            f.restype = i64
            f.argtypes = [vp]
        lib.vs_cube_fill.argtypes = [vp, vp, i64, i64, i64, i64, i64, i64, ctypes.c_int]
        lib.vs_layer_fill.argtypes = [u64, i64, i64, i64, vp, ctypes.c_int]
        lib.vs_cube_voxel.restype = ctypes.c_float
        lib.vs_cube_voxel.argtypes = [vp, i64, i64, i64]
        _cpu = lib
    return _cpu


def _cuda_lib():
    global _cuda
    if _cuda is None:
        lib = ctypes.CDLL(_build.build_cuda())
        i64, u64, vp = ctypes.c_int64, ctypes.c_uint64, ctypes.c_void_p
        lib.vs_dev_cube_create.restype = vp
        lib.vs_dev_cube_create.argtypes = [vp, i64, i64, i64]
        lib.vs_dev_cube_destroy.argtypes = [vp]
        lib.vs_dev_cube_fill.argtypes = [vp, vp, i64, i64, i64, i64, i64, i64, vp]
        lib.vs_dev_layer_fill.argtypes = [u64, i64, i64, i64, vp, vp]
        _cuda = lib
    return _cuda


def default_threads():
    import os
    try:
        return max(1, len(os.sched_getaffinity(0)))
    except AttributeError:
        return max(1, os.cpu_count() or 1)


class Cube:
    """A seeded synthetic spectral cube, evaluable anywhere (host box, device box, one voxel)."""

    def __init__(self, seed, nx, ny, nz, nsrc, ramp=0.0, kind=0):
        """kind SPECTRAL (0): N(0,1) noise + compact sources (+ spectral ramp); NBODY (1): the paper's other
        data family (Table 1 "Nbody"), a density cube that is zero except for nsrc extended halos."""
        self.seed, self.nx, self.ny, self.nz, self.nsrc, self.ramp = int(seed), int(nx), int(ny), int(nz), int(nsrc), float(ramp)
        self.kind = int(kind)
        self._h = _cpu_lib().vs_cube_create_kind(self.seed, self.nx, self.ny, self.nz, self.nsrc, self.ramp, self.kind)
        if not self._h:
            raise ValueError("bad cube parameters")
        self._d = None

    def __del__(self):
        try:
            if self._d:
                _cuda_lib().vs_dev_cube_destroy(self._d)
            if self._h:
                _cpu_lib().vs_cube_destroy(self._h)
        except Exception:
            pass

    @property
    def shape(self):
        return (self.nz, self.ny, self.nx)

    # -- host ---------------------------------------------------------------
    def fill_host(self, x0=0, y0=0, z0=0, sx=None, sy=None, sz=None, nthreads=None):
        sx = self.nx - x0 if sx is None else sx
        sy = self.ny - y0 if sy is None else sy
        sz = self.nz - z0 if sz is None else sz
        out = np.empty((sz, sy, sx), dtype=np.float32)
        _cpu_lib().vs_cube_fill(self._h, out.ctypes.data, x0, y0, z0, sx, sy, sz, nthreads or default_threads())
        return out

    def voxel(self, x, y, z):
        return float(_cpu_lib().vs_cube_voxel(self._h, x, y, z))

    def voxel_fn(self):
        """(function pointer, context) for the oracle's procedural-volume mode."""
        fn = ctypes.cast(_cpu_lib().vs_cube_voxel, ctypes.c_void_p).value
        return fn, self._h

    # -- device -------------------------------------------------------------
    def fill_device(self, dev_ptr, x0, y0, z0, sx, sy, sz, stream=0):
        lib = _cuda_lib()
        if self._d is None:
            c = _cpu_lib()
            self._d = lib.vs_dev_cube_create(self._h, c.vs_cube_nprof(self._h), c.vs_cube_ncell(self._h), c.vs_cube_nitems(self._h))
            if not self._d:
                raise RuntimeError("device upload of the synthetic-cube tables failed")
        rc = lib.vs_dev_cube_fill(self._d, dev_ptr, x0, y0, z0, sx, sy, sz, stream)
        if rc != 0:
            raise RuntimeError("vs_dev_cube_fill failed (%d)" % rc)


def layer_host(seed, layer, pix0, npix, nthreads=None):
    out = np.empty((npix, 4), dtype=np.float32)
    _cpu_lib().vs_layer_fill(int(seed), int(layer), int(pix0), int(npix), out.ctypes.data, nthreads or default_threads())
    return out


def layer_device(seed, layer, pix0, npix, dev_ptr, stream=0):
    rc = _cuda_lib().vs_dev_layer_fill(int(seed), int(layer), int(pix0), int(npix), dev_ptr, stream)
    if rc != 0:
        raise RuntimeError("vs_dev_layer_fill failed (%d)" % rc)


# ---------------------------------------------------------------------------
# seeded scalars (pure Python twin of vs_mix64, for cameras / permutations)
# ---------------------------------------------------------------------------
_M = (1 << 64) - 1


def mix64(x):
    x = (x + 0x9E3779B97F4A7C15) & _M
    x = ((x ^ (x >> 30)) * 0xBF58476D1CE4E5B9) & _M
    x = ((x ^ (x >> 27)) * 0x94D049BB133111EB) & _M
    return x ^ (x >> 31)


def u01(seed, stream, i):
    h = mix64((seed ^ (0xC0FFEE + stream * 0x100000001B3)) & _M ^ mix64(i))
    return ((h >> 11) + 0.5) / 9007199254740992.0


def permutation(seed, n):
    keys = [(mix64((seed * 1315423911 + i) & _M), i) for i in range(n)]
    keys.sort()
    return np.array([i for _, i in keys], dtype=np.int32)


# ---------------------------------------------------------------------------
# transfer functions (256-entry straight-alpha RGBA over [-3, 10])
# ---------------------------------------------------------------------------
TF_VMIN, TF_VMAX = -3.0, 10.0


def tf_ramp(n=256):
    """Primary: literal linear ramp, all four channels = u (BASELINE.json configs)."""
    u = np.linspace(0.0, 1.0, n, dtype=np.float64)
    return np.stack([u, u, u, u], axis=1).astype(np.float32)


def tf_density(n=256, toe=6):
    """For NBODY cubes over [0, NBODY_VMAX]: the ramp with a zero-opacity toe (entries < toe), so
    that empty space is exactly transparent and empty bricks can be skipped (R16)."""
    t = tf_ramp(n)
    t[:toe, 3] = 0.0
    return t


NBODY_VMAX = 20.0
SPECTRAL, NBODY = 0, 1


def tf_threshold(n=256, cut=0.5):
    """The usual way to look at a noisy spectral cube: the ramp with zero opacity below u = cut
    (value 3.5 sigma for cut = 0.5 over [-3, 10]), so that only the sources show."""
    t = tf_ramp(n)
    t[:int(round(cut * (n - 1))) + 1, 3] = 0.0
    return t


def tf_translucent(n=256):
    """Secondary: same colours, opacity u/64 per voxel (rays cross most of the cube)."""
    u = np.linspace(0.0, 1.0, n, dtype=np.float64)
    return np.stack([u, u, u, u / 64.0], axis=1).astype(np.float32)


# ---------------------------------------------------------------------------
# cameras: column-major float32[16], OpenGL clip conventions
# ---------------------------------------------------------------------------
def _colmajor(m):
    return np.ascontiguousarray(np.asarray(m, dtype=np.float64).T.reshape(16)).astype(np.float32)


def perspective(fovy_deg, aspect, near, far):
    f = 1.0 / math.tan(math.radians(fovy_deg) / 2.0)
    m = np.zeros((4, 4))
    m[0, 0] = f / aspect
    m[1, 1] = f
    m[2, 2] = (far + near) / (near - far)
    m[2, 3] = 2.0 * far * near / (near - far)
    m[3, 2] = -1.0
    return _colmajor(m)


def orthographic(half_w, half_h, near, far):
    m = np.eye(4)
    m[0, 0] = 1.0 / half_w
    m[1, 1] = 1.0 / half_h
    m[2, 2] = -2.0 / (far - near)
    m[2, 3] = -(far + near) / (far - near)
    return _colmajor(m)


def look_at(eye, centre, up):
    eye, centre, up = (np.asarray(v, dtype=np.float64) for v in (eye, centre, up))
    f = centre - eye
    f /= np.linalg.norm(f)
    s = np.cross(f, up)
    s /= np.linalg.norm(s)
    u = np.cross(s, f)
    m = np.eye(4)
    m[0, :3], m[1, :3], m[2, :3] = s, u, -f
    m[:3, 3] = -m[:3, :3] @ eye
    return _colmajor(m)


def quat_view(q, centre, dist):
    """view = T(0,0,-dist) * R(q) * T(-centre)."""
    w, x, y, z = q
    r = np.array([[1 - 2 * (y * y + z * z), 2 * (x * y - z * w), 2 * (x * z + y * w)],
                  [2 * (x * y + z * w), 1 - 2 * (x * x + z * z), 2 * (y * z - x * w)],
                  [2 * (x * z - y * w), 2 * (y * z + x * w), 1 - 2 * (x * x + y * y)]])
    m = np.eye(4)
    m[:3, :3] = r
    m[:3, 3] = -r @ np.asarray(centre, dtype=np.float64) + np.array([0.0, 0.0, -dist])
    return _colmajor(m)


def seeded_quat(seed, i):
    """Uniform random rotation (Shoemake) from the seeded hash."""
    u1, u2, u3 = u01(seed, 11, i), u01(seed, 12, i), u01(seed, 13, i)
    a, b = math.sqrt(1 - u1), math.sqrt(u1)
    return (b * math.cos(2 * math.pi * u3), a * math.sin(2 * math.pi * u2),
            a * math.cos(2 * math.pi * u2), b * math.sin(2 * math.pi * u3))


class Framing:
    """DESIGN.md camera: volume centred, bounding sphere R, fovy 40 deg, eye at 1.05 R / sin 20 deg."""

    def __init__(self, nx, ny, nz, width, height):
        self.centre = (nx / 2.0, ny / 2.0, nz / 2.0)
        self.R = 0.5 * math.sqrt(nx * nx + ny * ny + nz * nz)
        self.aspect = width / float(height)
        self.dist = 1.05 * self.R / math.sin(math.radians(20.0))
        self.near, self.far = self.dist - 1.01 * self.R, self.dist + 1.01 * self.R

    def proj(self, ortho=False):
        if ortho:
            hh = 1.05 * self.R
            return orthographic(hh * self.aspect, hh, self.near, self.far)
        return perspective(40.0, self.aspect, self.near, self.far)

    def turntable(self, k, nviews=36, elevation_deg=20.0):
        """k-th view of a turntable about the spectral (z) axis, shown vertical."""
        az = 2.0 * math.pi * k / nviews
        el = math.radians(elevation_deg)
        c = np.asarray(self.centre)
        eye = c + self.dist * np.array([math.cos(el) * math.cos(az), math.cos(el) * math.sin(az), math.sin(el)])
        return look_at(eye, c, (0.0, 0.0, 1.0))

    def seeded(self, seed, k):
        return quat_view(seeded_quat(seed, k), self.centre, self.dist)


# ---------------------------------------------------------------------------
# the five BASELINE.json configurations (shape/statistics only)
# ---------------------------------------------------------------------------
CONFIGS = {
    "c0": dict(nx=64, ny=64, nz=64, brick=64, ghost=1, nsrc=8, ramp=0.0, width=256, height=256, step=0.5),
    "c1": dict(nx=512, ny=512, nz=512, brick=256, ghost=1, nsrc=200, ramp=0.0, width=1024, height=1024, step=0.5),
    "c2": dict(nx=1024, ny=1024, nz=1024, brick=256, ghost=1, nsrc=2000, ramp=1.0, width=1920, height=1080, step=0.5),
    "c3": dict(nx=4096, ny=4096, nz=1536, brick=512, ghost=1, nsrc=50000, ramp=0.0, width=1920, height=1080, step=1.0),
    # row f4 (not a BASELINE.json config): the paper's other data family (Table 1 "Nbody" 1024^3, "scaled Nbody"
    # 2600^3): a 2048^3 density cube (34 GB), zero except for 200 extended halos, in 512 bricks of 256^3
    # not a BASELINE.json config: config 3 at half scale (the same voxels-per-pixel ratio, bricks of 256^3: 8x8x3 grid, 26 GB),
    # small enough for the texture arm's second copy of the bricks - the sparse-sampling regime for BOTH samplers
    "s3": dict(nx=2048, ny=2048, nz=768, brick=256, ghost=1, nsrc=6250, ramp=0.0, width=960, height=540, step=1.0),
    "n1": dict(nx=2048, ny=2048, nz=2048, brick=256, ghost=1, nsrc=200, ramp=0.0, width=1920, height=1080, step=0.5, kind=1),
}


def config_cube(name):
    c = CONFIGS[name]
    k = int(name[1:]) + {"n": 10, "s": 20}.get(name[0], 0)
    return Cube(BASE_SEED + k, c["nx"], c["ny"], c["nz"], c["nsrc"], c["ramp"], c.get("kind", 0))
