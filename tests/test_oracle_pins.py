"""Pins for the CPU oracle (oracle/vr_oracle.c): closed forms, invariants, special cases and an
independent brute-force numpy renderer. None of these call the CUDA path. Citations are
PAPER.md lines; R# are the readings of DESIGN.md."""
import math
import os

import numpy as np
import pytest

import oracle
import synth

GOLD = os.path.join(os.path.dirname(__file__), "golden")


# --------------------------------------------------------------------------- helpers
def ortho_along_z(nx, ny, nz):
    """Axis-aligned orthographic camera looking along +z, one pixel per voxel column.
    Pixel (i, j) looks down the column x = nx-1-i, y = j (the look-at basis mirrors x)."""
    view = synth.look_at((nx / 2.0, ny / 2.0, -10.0), (nx / 2.0, ny / 2.0, 0.0), (0.0, 1.0, 0.0))
    proj = synth.orthographic(nx / 2.0, ny / 2.0, 1.0, 30.0 + nz)
    return view, proj


def const_tf(rgb, a, n=4):
    t = np.zeros((n, 4), dtype=np.float32)
    t[:, :3] = rgb
    t[:, 3] = a
    return t


def mats(view, proj):
    V = np.asarray(view, dtype=np.float64).reshape(4, 4).T
    P = np.asarray(proj, dtype=np.float64).reshape(4, 4).T
    return V, P


def ray_np(view, proj, W, H, i, j):
    """Independent statement of R1/R2 with numpy's own inverse."""
    V, P = mats(view, proj)
    Minv = np.linalg.inv(P @ V)
    x, y = 2 * (i + 0.5) / W - 1, 2 * (j + 0.5) / H - 1
    a = Minv @ np.array([x, y, -1.0, 1.0])
    b = Minv @ np.array([x, y, 1.0, 1.0])
    a, b = a[:3] / a[3], b[:3] / b[3]
    L = np.linalg.norm(b - a)
    return a, (b - a) / L, L


def chord_np(o, d, L, n):
    """Independent clip of the segment o + t d, t in [0, L], against [0,n] (Liang-Barsky)."""
    t0, t1 = 0.0, L
    for a in range(3):
        if abs(d[a]) < 1e-300:
            if o[a] < 0 or o[a] > n[a]:
                return None
            continue
        ta, tb = (0 - o[a]) / d[a], (n[a] - o[a]) / d[a]
        t0, t1 = max(t0, min(ta, tb)), min(t1, max(ta, tb))
    return (t0, t1) if t1 > t0 else None


def brute_force_render(data, tf, vmin, vmax, view, proj, W, H, step, mode):
    """Independent, unbricked, global renderer written from the definitions (numpy/python)."""
    nz, ny, nx = data.shape
    n = (nx, ny, nz)
    lut = np.asarray(tf, dtype=np.float64)
    N = lut.shape[0]
    img = np.zeros((H, W, 4))

    def vox(ix, iy, iz):
        return float(data[min(max(iz, 0), nz - 1), min(max(iy, 0), ny - 1), min(max(ix, 0), nx - 1)])

    def tri(p):
        q = [p[0] - 0.5, p[1] - 0.5, p[2] - 0.5]
        i0 = [math.floor(c) for c in q]
        f = [q[a] - i0[a] for a in range(3)]
        acc = 0.0
        for dz in (0, 1):
            for dy in (0, 1):
                for dx in (0, 1):
                    w = (f[0] if dx else 1 - f[0]) * (f[1] if dy else 1 - f[1]) * (f[2] if dz else 1 - f[2])
                    acc += w * vox(i0[0] + dx, i0[1] + dy, i0[2] + dz)
        return acc

    def lut_at(v):
        u = min(max((v - vmin) / (vmax - vmin), 0.0), 1.0)
        xs = np.arange(N) / (N - 1.0)
        return np.array([np.interp(u, xs, lut[:, c]) for c in range(4)])

    for j in range(H):
        for i in range(W):
            o, d, L = ray_np(view, proj, W, H, i, j)
            ch = chord_np(o, d, L, n)
            if ch is None:
                continue
            t0, t1 = ch
            K = int(math.ceil((t1 - t0) / step))
            C, A, m, took = np.zeros(3), 0.0, -np.inf, 0
            for k in range(K):
                a0, a1 = t0 + k * step, min(t0 + (k + 1) * step, t1)
                if a1 <= a0:
                    continue
                v = tri(o + 0.5 * (a0 + a1) * d)
                took += 1
                if mode == oracle.MIP:
                    m = max(m, v)
                else:
                    rgba = lut_at(v)
                    al = 1 - (1 - rgba[3]) ** (a1 - a0)
                    C += (1 - A) * al * rgba[:3]
                    A += (1 - A) * al
            if mode == oracle.MIP:
                if took:
                    img[j, i, :3] = lut_at(m)[:3]
                    img[j, i, 3] = 1.0
            else:
                img[j, i, :3], img[j, i, 3] = C, A
    return img


def small_noise(nx, ny, nz, seed=7, nsrc=3):
    return synth.Cube(seed, nx, ny, nz, nsrc).fill_host(nthreads=1)


# --------------------------------------------------------------------------- golden (paper's printed values)
def test_table1_sizes_pin_float32_voxels():
    """dims x 4 B reproduce the printed file sizes => float32 voxels."""
    for line in open(os.path.join(GOLD, "table1_datasets.txt")):
        if line.startswith("#") or not line.strip():
            continue
        name, nx, ny, nz, gb = [s.strip() for s in line.split("|")]
        gib = int(nx) * int(ny) * int(nz) * np.dtype(np.float32).itemsize / 2.0 ** 30
        assert abs(gib - float(gb)) <= 0.7, (name, gib)           # printed values are rounded
        assert abs(gib * 2 - float(gb)) > 0.7 * float(gb) / 4     # float64 would not fit the table


def test_subframe_message_is_one_float_per_pixel():
    """4 MB per 1024x1024 frame => 4 B/pixel (MIP scalar sub-image, row a8)."""
    for line in open(os.path.join(GOLD, "subframe_message.txt")):
        if line.startswith("#") or not line.strip():
            continue
        w, h, mb = [float(s) for s in line.split("|")]
        assert w * h * np.dtype(np.float32).itemsize == mb * 2 ** 20


# --------------------------------------------------------------------------- pin 1: homogeneous cube
@pytest.mark.parametrize("ortho", [False, True])
def test_homogeneous_cube_closed_form(ortho):
    """north_star: opacity 1-exp(-sigma L) = 1-(1-a)^L along every ray; exact by R5."""
    nx, ny, nz = 12, 9, 15
    a, rgb = float(np.float32(0.07)), (0.2, 0.5, 0.9)   # the LUT stores float32
    data = np.full((nz, ny, nx), 1.25, dtype=np.float32)
    W = H = 24
    fr = synth.Framing(nx, ny, nz, W, H)
    for bricks in (64, 5):
        vol = oracle.Volume(nx, ny, nz, bricks, 1, data=data)
        vol.set_transfer_function(const_tf(rgb, a), -3, 10)
        vol.set_early_termination(2.0)
        for k in range(3):
            view, proj = fr.seeded(99, k), fr.proj(ortho)
            img = vol.render(view, proj, W, H, 0.37, oracle.ALPHA, nthreads=2)["image"]
            nhit = 0
            for j in range(0, H, 3):
                for i in range(0, W, 3):
                    o, d, L = ray_np(view, proj, W, H, i, j)
                    ch = chord_np(o, d, L, (nx, ny, nz))
                    A = 0.0 if ch is None else 1 - (1 - a) ** (ch[1] - ch[0])
                    nhit += ch is not None
                    assert abs(img[j, i, 3] - A) < 1e-12
                    np.testing.assert_allclose(img[j, i, :3], A * np.array(rgb, dtype=np.float32).astype(np.float64), atol=1e-12)
            assert nhit > 10


def test_camera_inside_volume_starts_at_near_plane():
    """R2: path length is measured from the near plane when the camera is inside the cube."""
    n = 20
    data = np.zeros((n, n, n), dtype=np.float32)
    a = float(np.float32(0.1))
    vol = oracle.Volume(n, n, n, 8, 1, data=data)
    vol.set_transfer_function(const_tf((1, 1, 1), a), -3, 10)
    vol.set_early_termination(2.0)
    view = synth.look_at((10.0, 10.0, 4.0), (10.0, 10.0, 20.0), (0.0, 1.0, 0.0))
    proj = synth.perspective(30.0, 1.0, 2.0, 100.0)
    W = H = 9
    img = vol.render(view, proj, W, H, 0.5, oracle.ALPHA)["image"]
    o, d, L = ray_np(view, proj, W, H, 4, 4)          # centre pixel: straight along +z
    assert abs(o[2] - 6.0) < 1e-5 and abs(d[2] - 1.0) < 1e-9
    assert abs(img[4, 4, 3] - (1 - (1 - a) ** (20.0 - o[2]))) < 1e-12


# --------------------------------------------------------------------------- pin 2: single bright voxel
def test_single_voxel_tent_mip():
    """R3/R11: the interpolant of one bright voxel is a tent; axis-aligned rays sampling the
    centre plane see V (1-|dx|)(1-|dy|)."""
    n, V = 8, 8.0                     # n/2 is a power of two: the float32 matrices are exact
    data = np.zeros((n, n, n), dtype=np.float32)
    c = (4, 3, 5)                     # (x, y, z) index of the bright voxel
    data[c[2], c[1], c[0]] = V
    ident = np.zeros((256, 4), dtype=np.float32)
    ident[:, 0] = np.linspace(0, 1, 256)
    ident[:, 3] = 1
    sub = 4                           # 4 x 4 pixels per voxel => lateral offsets +-1/8, +-3/8 ...
    W = H = n * sub
    view, proj = ortho_along_z(n, n, n)
    for brick in (16, 4):
        vol = oracle.Volume(n, n, n, brick, 1, data=data)
        vol.set_transfer_function(ident, 0.0, 10.0)
        img = vol.render(view, proj, W, H, 1.0, oracle.MIP)["image"]
        for j in range(H):
            for i in range(W):
                x = n - (i + 0.5) / sub            # world x of the ray (mirrored basis)
                y = (j + 0.5) / sub
                tent = V * max(0.0, 1 - abs(x - (c[0] + 0.5))) * max(0.0, 1 - abs(y - (c[1] + 0.5)))
                want = np.interp(tent / 10.0, np.arange(256) / 255.0, ident[:, 0].astype(np.float64))
                assert abs(img[j, i, 0] - want) < 1e-12 and abs(want - tent / 10.0) < 1e-7
                assert img[j, i, 3] == 1.0


def test_centre_pixel_hits_volume_centre_and_mirror():
    """R1: a symmetric view puts the volume centre on the centre of the frame; mirroring the
    camera's x axis mirrors the image."""
    n = 9
    data = np.zeros((n, n, n), dtype=np.float32)
    data[4, 4, 4] = 5.0
    data[2, 6, 1] = 3.0               # an asymmetric marker
    vol = oracle.Volume(n, n, n, 4, 1, data=data)
    vol.set_transfer_function(synth.tf_ramp(), -3, 10)
    W = H = 15
    fr = synth.Framing(n, n, n, W, H)
    view, proj = fr.turntable(0), fr.proj(False)
    img = vol.render(view, proj, W, H, 0.25, oracle.MIP)["image"]
    jm, im = np.unravel_index(np.argmax(img[:, :, 0]), (H, W))
    assert (jm, im) == (H // 2, W // 2)
    flip = np.diag([-1.0, 1.0, 1.0, 1.0])
    P = np.asarray(proj, dtype=np.float64).reshape(4, 4).T
    proj_m = np.ascontiguousarray((flip @ P).T.reshape(16)).astype(np.float32)
    img_m = vol.render(view, proj_m, W, H, 0.25, oracle.MIP)["image"]
    np.testing.assert_allclose(img_m, img[:, ::-1, :], atol=1e-12)
    assert np.abs(img - img[:, ::-1, :]).max() > 1e-3


# --------------------------------------------------------------------------- pin 3: axis-aligned orthographic
def test_axis_aligned_ortho_mip_is_column_max_and_alpha_closed_form():
    """north_star: axis-aligned orthographic MIP == per-column max; ALPHA == the column's
    front-to-back product form (samples fall on voxel centres, w = 1). All d_a = 0 on two axes (R4)."""
    nx, ny, nz = 8, 16, 13            # nx/2, ny/2 powers of two: the float32 matrices are exact
    data = small_noise(nx, ny, nz)
    view, proj = ortho_along_z(nx, ny, nz)
    tf = synth.tf_translucent()
    tf[:, 3] *= 20.0
    tf = np.clip(tf, 0, 1).astype(np.float32)
    vmin, vmax = -3.0, 10.0
    for brick in (32, 4):
        vol = oracle.Volume(nx, ny, nz, brick, 1, data=data)
        vol.set_transfer_function(tf, vmin, vmax)
        vol.set_early_termination(2.0)
        mip = vol.render(view, proj, nx, ny, 1.0, oracle.MIP)["image"]
        alp = vol.render(view, proj, nx, ny, 1.0, oracle.ALPHA)["image"]
        lut = tf.astype(np.float64)
        xs = np.arange(256) / 255.0
        for j in range(ny):
            for i in range(nx):
                col = data[:, j, nx - 1 - i].astype(np.float64)
                u = np.clip((col.max() - vmin) / (vmax - vmin), 0, 1)
                assert abs(mip[j, i, 0] - np.interp(u, xs, lut[:, 0])) < 1e-12
                uu = np.clip((col - vmin) / (vmax - vmin), 0, 1)
                al = np.interp(uu, xs, lut[:, 3])
                cr = np.interp(uu, xs, lut[:, 0])
                T = np.concatenate([[1.0], np.cumprod(1 - al)[:-1]])
                assert abs(alp[j, i, 3] - (1 - np.prod(1 - al))) < 1e-12
                assert abs(alp[j, i, 0] - np.sum(T * al * cr)) < 1e-12


# --------------------------------------------------------------------------- pin 4: 1 brick == N bricks
@pytest.mark.parametrize("mode", [oracle.ALPHA, oracle.MIP])
def test_one_brick_equals_n_bricks_ragged(mode):
    """north_star / R3: with ghost >= 1 and ERT off the image does not depend on the bricking,
    ragged grids included; no fetch leaves a padded brick. ghost = 0 must differ (seams)."""
    nx, ny, nz = 19, 11, 13
    data = small_noise(nx, ny, nz)
    W, H = 32, 24
    fr = synth.Framing(nx, ny, nz, W, H)
    one = oracle.Volume(nx, ny, nz, 64, 1, data=data)
    many = oracle.Volume(nx, ny, nz, 5, 1, data=data)
    seam = oracle.Volume(nx, ny, nz, 5, 0, data=data)
    assert many.nbricks == 4 * 3 * 3
    for v in (one, many, seam):
        v.set_transfer_function(synth.tf_ramp(), -3, 10)
        v.set_early_termination(2.0)
    worst_seam = 0.0
    for k, ortho in ((0, False), (1, True), (2, False)):
        view, proj = fr.seeded(5, k), fr.proj(ortho)
        a = one.render(view, proj, W, H, 0.5, mode)
        b = many.render(view, proj, W, H, 0.5, mode)
        s = seam.render(view, proj, W, H, 0.5, mode)
        assert np.abs(a["image"] - b["image"]).max() < 1e-12
        assert np.array_equal(a["counts"][..., 1], b["counts"][..., 1])      # same schedule
        worst_seam = max(worst_seam, np.abs(a["image"] - s["image"]).max())
    assert one.ghost_violations() == 0 and many.ghost_violations() == 0
    assert seam.ghost_violations() > 0 and worst_seam > 1e-3


def test_oracle_bricks_are_edge_replicated_copies():
    """a1 / R3: a padded brick equals the clamped-index gather of the source."""
    nx, ny, nz = 10, 7, 6
    data = small_noise(nx, ny, nz)
    g, B = 2, 4
    vol = oracle.Volume(nx, ny, nz, B, g, data=data)
    b = 0
    for bz in range(2):
        for by in range(2):
            for bx in range(3):
                got = vol.brick_data(b)
                zs = np.clip(np.arange(bz * B - g, min(bz * B + B, nz) + g), 0, nz - 1)
                ys = np.clip(np.arange(by * B - g, min(by * B + B, ny) + g), 0, ny - 1)
                xs = np.clip(np.arange(bx * B - g, min(bx * B + B, nx) + g), 0, nx - 1)
                assert np.array_equal(got, data[np.ix_(zs, ys, xs)])
                b += 1


# --------------------------------------------------------------------------- pin 5: ERT bound
def test_ert_within_one_minus_tau():
    """R8: brick-local termination at tau changes a channel by at most (1 - tau)."""
    nx = ny = nz = 24
    data = small_noise(nx, ny, nz)
    W = H = 24
    fr = synth.Framing(nx, ny, nz, W, H)
    view, proj = fr.turntable(3), fr.proj(False)
    for tau in (0.99, 0.9):
        vol = oracle.Volume(nx, ny, nz, 8, 1, data=data)
        vol.set_transfer_function(synth.tf_ramp(), -3, 10)
        vol.set_early_termination(2.0)
        off = vol.render(view, proj, W, H, 0.5, oracle.ALPHA)
        vol.set_early_termination(tau)
        on = vol.render(view, proj, W, H, 0.5, oracle.ALPHA)
        diff = np.abs(off["image"] - on["image"]).max()
        assert 0 < diff <= (1 - tau) + 1e-12
        assert on["counts"][..., 0].sum() < off["counts"][..., 0].sum()
        assert np.array_equal(on["counts"][..., 1], off["counts"][..., 1])


# --------------------------------------------------------------------------- pin 6/7: ordering
def test_mip_is_order_independent_alpha_is_not():
    """MIP composites in arbitrary order; `over` does not."""
    nx, ny, nz = 16, 16, 16
    data = small_noise(nx, ny, nz)
    W = H = 16
    fr = synth.Framing(nx, ny, nz, W, H)
    view, proj = fr.seeded(1, 0), fr.proj(False)
    vol = oracle.Volume(nx, ny, nz, 4, 1, data=data)
    vol.set_transfer_function(synth.tf_ramp(), -3, 10)
    vol.set_early_termination(2.0)
    mip0 = vol.render(view, proj, W, H, 0.5, oracle.MIP)["image"]
    alp0 = vol.render(view, proj, W, H, 0.5, oracle.ALPHA)["image"]
    vol.set_order_override(synth.permutation(3, vol.nbricks))
    assert np.array_equal(vol.render(view, proj, W, H, 0.5, oracle.MIP)["image"], mip0)
    assert np.abs(vol.render(view, proj, W, H, 0.5, oracle.ALPHA)["image"] - alp0).max() > 1e-3


@pytest.mark.parametrize("ortho", [False, True])
def test_visibility_order_contains_every_ray_order(ortho):
    """R9/R10: the global order is a permutation; every ray's t_in order is a subsequence of it;
    consecutive bricks on a ray share a face; bricks holding samples are on the ray's list;
    no brick holds samples for a pixel outside its rendering rectangle."""
    nx, ny, nz = 19, 11, 13
    data = small_noise(nx, ny, nz)
    W, H = 20, 16
    fr = synth.Framing(nx, ny, nz, W, H)
    vol = oracle.Volume(nx, ny, nz, 5, 1, data=data)
    vol.set_transfer_function(synth.tf_ramp(), -3, 10)
    vol.set_early_termination(2.0)
    pix = np.array([(i, j) for j in range(H) for i in range(W)], dtype=np.int32)
    views = [fr.seeded(11, k) for k in range(4)]
    # plus an eye inside the brick grid's span on one axis (distance-0 slab)
    views.append(synth.look_at((9.5, 40.0, 6.0), (9.5, 5.0, 6.0), (0, 0, 1)))
    for view in views:
        proj = fr.proj(ortho) if view is not views[-1] else synth.perspective(50.0, W / H, 1.0, 200.0)
        order = vol.brick_order(view, proj)
        assert sorted(order.tolist()) == list(range(vol.nbricks))
        pos = np.empty(vol.nbricks, dtype=np.int64)
        pos[order] = np.arange(vol.nbricks)
        counts, lists, graz = vol.ray_bricks(view, proj, W, H, pix, maxlen=16)
        res = vol.render(view, proj, W, H, 0.5, oracle.MIP, pixels=pix, want_sub=True)
        rects = vol.rects(view, proj, W, H)
        hit_any = 0
        for q in range(len(pix)):
            if graz[q]:
                continue
            lst = lists[q, :counts[q]]
            assert np.all(np.diff(pos[lst]) > 0), "ray order must embed in the global order"
            for b0, b1 in zip(lst[:-1], lst[1:]):
                c0 = np.array([b0 % 4, (b0 // 4) % 3, b0 // 12])
                c1 = np.array([b1 % 4, (b1 // 4) % 3, b1 // 12])
                assert np.abs(c0 - c1).sum() == 1, "consecutive bricks share a face"
            holders = np.nonzero(res["sub"][q, :, 1] > 0)[0]
            assert set(holders.tolist()) <= set(lst.tolist())
            assert res["sub"][q, :, 1].sum() == res["counts"][q, 0] == res["counts"][q, 1]
            i, j = pix[q]
            for b in holders:
                x0, y0, x1, y1 = rects[b]
                assert x0 <= i < x1 and y0 <= j < y1
            hit_any += len(lst) > 0
        assert hit_any > 50


def test_visibility_order_ragged_grid_close_eyes():
    """R9 on a strongly ragged grid (slabs 5,5,1 / 4,3 / 6,2) with eyes close to and inside the
    volume: slab-distance ranks stay valid where centre-distance sorting does not."""
    nx, ny, nz = 11, 7, 8
    vol = oracle.Volume(nx, ny, nz, 5, 1, data=np.zeros((nz, ny, nx), dtype=np.float32))
    g = (3, 2, 2)
    W = H = 24
    pix = np.array([(i, j) for j in range(H) for i in range(W)], dtype=np.int32)
    proj = synth.perspective(70.0, 1.0, 0.05, 60.0)
    checked = 0
    for k in range(60):
        eye = np.array([synth.u01(5, a, k) * (n + 6.0) - 3.0 for a, n in enumerate((nx, ny, nz))])
        tgt = np.array([synth.u01(6, a, k) * n for a, n in enumerate((nx, ny, nz))])
        if np.linalg.norm(tgt - eye) < 0.5:
            continue
        view = synth.look_at(eye, tgt, (0.123, 0.456, 0.881))
        order = vol.brick_order(view, proj)
        pos = np.empty(vol.nbricks, dtype=np.int64)
        pos[order] = np.arange(vol.nbricks)
        counts, lists, graz = vol.ray_bricks(view, proj, W, H, pix, maxlen=16)
        for q in range(len(pix)):
            if graz[q] or counts[q] < 2:
                continue
            assert np.all(np.diff(pos[lists[q, :counts[q]]]) > 0)
            checked += 1
    assert checked > 5000


# --------------------------------------------------------------------------- pin 8: convergence
def test_step_halving_converges():
    """R5: midpoint rule on a smooth field; halving the step shrinks the error."""
    n = 24
    z, y, x = np.meshgrid(*(np.arange(n) + 0.5,) * 3, indexing="ij")
    data = (2.0 + 3.0 * np.sin(x / 5.0) * np.cos(y / 6.0) + 2.0 * np.sin(z / 4.0)).astype(np.float32)
    W = H = 12
    fr = synth.Framing(n, n, n, W, H)
    view, proj = fr.seeded(2, 1), fr.proj(False)
    vol = oracle.Volume(n, n, n, 8, 1, data=data)
    tf = synth.tf_translucent()
    tf[:, 3] *= 8
    vol.set_transfer_function(tf.astype(np.float32), -3, 10)
    vol.set_early_termination(2.0)
    ref = vol.render(view, proj, W, H, 1.0 / 64, oracle.ALPHA)["image"]
    errs = [np.abs(vol.render(view, proj, W, H, s, oracle.ALPHA)["image"] - ref).max() for s in (1.0, 0.5, 0.25)]
    assert errs[0] > errs[1] > errs[2] > 0
    assert errs[2] < errs[0] / 6.0


# --------------------------------------------------------------------------- pin 9: brute force
@pytest.mark.parametrize("mode", [oracle.ALPHA, oracle.MIP])
@pytest.mark.parametrize("ortho", [False, True])
def test_against_independent_brute_force_renderer(mode, ortho):
    """Tiny inputs (<= 16^3, <= 16^2 pixels): the bricked C oracle equals an unbricked numpy
    renderer written separately from the definitions."""
    nx, ny, nz = 13, 9, 11
    data = small_noise(nx, ny, nz, seed=21)
    W, H = 12, 10
    fr = synth.Framing(nx, ny, nz, W, H)
    tf = synth.tf_ramp()
    tf[:, 1] = tf[::-1, 1]
    tf[:, 3] *= 0.3
    view, proj = fr.seeded(4, 2), fr.proj(ortho)
    vol = oracle.Volume(nx, ny, nz, 4, 1, data=data)
    vol.set_transfer_function(tf, -2.0, 6.0)
    vol.set_early_termination(2.0)
    got = vol.render(view, proj, W, H, 0.4, mode)["image"]
    want = brute_force_render(data, tf, -2.0, 6.0, view, proj, W, H, 0.4, mode)
    assert np.abs(got - want).max() < 1e-9
    assert (want[..., 3] > 0).sum() > 20


# --------------------------------------------------------------------------- TF special cases (R7)
def test_transfer_function_special_cases():
    n = 12
    data = small_noise(n, n, n)
    W = H = 10
    fr = synth.Framing(n, n, n, W, H)
    view, proj = fr.seeded(8, 0), fr.proj(False)
    vol = oracle.Volume(n, n, n, 5, 1, data=data)
    vol.set_early_termination(2.0)
    # a = 0: fully transparent frame
    vol.set_transfer_function(const_tf((1, 1, 1), 0.0), -3, 10)
    assert np.abs(vol.render(view, proj, W, H, 0.5, oracle.ALPHA)["image"]).max() == 0.0
    # a = 1: the first sample's colour exactly, opacity 1
    tf = synth.tf_ramp()
    tf[:, 3] = 1.0
    vol.set_transfer_function(tf, -3, 10)
    img = vol.render(view, proj, W, H, 0.5, oracle.ALPHA)["image"]
    hit = img[..., 3] > 0
    assert hit.sum() > 10 and np.all(img[hit][:, 3] == 1.0)
    one = oracle.Volume(n, n, n, 64, 1, data=data)
    one.set_transfer_function(tf, -3, 10)
    one.set_early_termination(0.5)         # stops after the first sample
    assert np.abs(one.render(view, proj, W, H, 0.5, oracle.ALPHA)["image"] - img).max() < 1e-12
    # constant colour: C = A c
    c = np.array([0.3, 0.6, 0.1], dtype=np.float32)
    tf2 = synth.tf_ramp()
    tf2[:, :3] = c
    vol.set_transfer_function(tf2, -3, 10)
    img = vol.render(view, proj, W, H, 0.5, oracle.ALPHA)["image"]
    np.testing.assert_allclose(img[..., :3], img[..., 3:4] * c.astype(np.float64), atol=1e-12)


# --------------------------------------------------------------------------- compositing (R15)
def test_composite_over_is_associative_and_matches_numpy():
    W, H, n = 13, 9, 6
    rects = [(0, 0, W, H), (2, 1, 9, 7), (5, 0, 13, 4), (0, 3, 6, 9), (4, 4, 5, 5), (1, 1, 12, 8)]
    layers = []
    for l, r in enumerate(rects):
        layers.append(synth.layer_host(77, l, 0, (r[2] - r[0]) * (r[3] - r[1])).reshape(r[3] - r[1], r[2] - r[0], 4))
    order = synth.permutation(9, n)
    got = oracle.composite(layers, rects, order, W, H)
    want = np.zeros((H, W, 4))
    for l in order:
        r = rects[l]
        full = np.zeros((H, W, 4))
        full[r[1]:r[3], r[0]:r[2]] = layers[l]
        want += (1 - want[..., 3:4]) * full
    assert np.abs(got - want).max() < 1e-15
    # associativity: composite the two halves separately, then merge
    h1 = oracle.composite([layers[l] for l in order[:3]], [rects[l] for l in order[:3]], np.arange(3), W, H)
    h2 = oracle.composite([layers[l] for l in order[3:]], [rects[l] for l in order[3:]], np.arange(3), W, H)
    merged = h1 + (1 - h1[..., 3:4]) * h2
    assert np.abs(merged - got).max() < 1e-12


# --------------------------------------------------------------------------- data range (row f1, R16)
def test_brick_minmax_planted_extremes_and_ghost_cells():
    """PAPER.md:146 local minimum and maximum: per brick over its ghost-padded cells. A voxel on
    a brick face belongs to the neighbour's ghost layer, so BOTH bricks see it; a voxel two
    cells inside does not leak; the global range is the range of the volume."""
    nx, ny, nz, B = 12, 8, 8, 4                      # 3 x 2 x 2 bricks
    data = np.zeros((nz, ny, nx), dtype=np.float32)
    data[1, 1, 3] = 7.5                              # last core cell of brick 0 along x -> ghost of brick 1
    data[1, 1, 4] = -2.25                            # first core cell of brick 1 -> ghost of brick 0
    data[6, 6, 10] = 9.0                             # two cells inside brick 11: nobody else sees it
    vol = oracle.Volume(nx, ny, nz, B, 1, data=data)
    assert vol.brick_minmax(0) == (np.float32(-2.25), np.float32(7.5))
    assert vol.brick_minmax(1) == (np.float32(-2.25), np.float32(7.5))
    assert vol.brick_minmax(2) == (np.float32(0.0), np.float32(0.0))
    assert vol.brick_minmax(11) == (np.float32(0.0), np.float32(9.0))
    for b in (3, 4, 5, 6, 7, 8, 9, 10):
        assert vol.brick_minmax(b) == (np.float32(0.0), np.float32(0.0)), b
    assert vol.brick_minmax(-1) == (np.float32(-2.25), np.float32(9.0))
    # ghost = 0: the face voxels stay private
    vol0 = oracle.Volume(nx, ny, nz, B, 0, data=data)
    assert vol0.brick_minmax(0) == (np.float32(0.0), np.float32(7.5))
    assert vol0.brick_minmax(1) == (np.float32(-2.25), np.float32(0.0))


@pytest.mark.parametrize("ghost", [0, 1, 2])
def test_brick_minmax_brute_force_ragged(ghost):
    """Against numpy's edge padding (an independent statement of the clamp rule) on a ragged grid,
    dense and procedural storage."""
    cube = synth.Cube(31, 11, 9, 7, 2)
    data = cube.fill_host()
    B = 4
    pad = np.pad(data, ghost, mode="edge")
    for vol in (oracle.Volume(11, 9, 7, B, ghost, data=data), oracle.Volume(11, 9, 7, B, ghost, voxel_fn=cube.voxel_fn())):
        b = 0
        for bz in range(2):
            for by in range(3):
                for bx in range(3):
                    x0, y0, z0 = bx * B, by * B, bz * B
                    x1, y1, z1 = min(x0 + B, 11), min(y0 + B, 9), min(z0 + B, 7)
                    box = pad[z0:z1 + 2 * ghost, y0:y1 + 2 * ghost, x0:x1 + 2 * ghost]
                    assert vol.brick_minmax(b) == (box.min(), box.max()), b
                    b += 1
        assert vol.brick_minmax(-1) == (data.min(), data.max())


def test_transparent_brick_rule_boundaries():
    """R16 on constant bricks: entry range [I(min)-1, I(max)+2] must be all zero-alpha."""
    n = 101                                          # table coordinate = value when vmin, vmax = 0, 100
    def vol_of(value, alpha_nonzero):
        v = oracle.Volume(4, 4, 4, 4, 1, data=np.full((4, 4, 4), value, dtype=np.float32))
        tf = np.zeros((n, 4), dtype=np.float32)
        tf[:, :3] = 0.5
        tf[list(alpha_nonzero), 3] = 0.25
        v.set_transfer_function(tf, 0.0, 100.0)
        return v
    hi = range(50, n)                                # opaque from entry 50 up
    assert vol_of(47.5, hi).brick_transparent(0)     # I = 47 -> entries 46..49
    assert not vol_of(48.5, hi).brick_transparent(0)  # I = 48 -> entries 47..50
    assert not vol_of(60.0, hi).brick_transparent(0)
    lo = range(0, 11)                                # opaque up to entry 10
    assert not vol_of(11.5, lo).brick_transparent(0)  # I = 11 -> entries 10..13
    assert vol_of(12.5, lo).brick_transparent(0)     # I = 12 -> entries 11..14
    assert vol_of(-5.0, hi).brick_transparent(0)     # clamped below the table
    assert not vol_of(500.0, hi).brick_transparent(0)  # clamped above: I = n-2 -> entries n-3..n-1
    assert vol_of(500.0, lo).brick_transparent(0)


def test_transparent_bricks_render_exactly_nothing():
    """The point of R16: skipping a transparent brick changes no output bit, because all of its
    samples classify to alpha 0 - its sub-image is exactly zero for every ray (ALPHA)."""
    nx, ny, nz, B = 24, 16, 16, 8                    # 3 x 2 x 2 bricks
    data = synth.Cube(5, nx, ny, nz, 3).fill_host()
    faint = np.clip(data, -2.9, -1.2)
    for (bx, by, bz) in ((0, 0, 0), (2, 1, 0), (1, 0, 1)):   # these bricks (with a margin for the ghosts) hold faint values only
        x0, y0, z0 = max(bx * B - 1, 0), max(by * B - 1, 0), max(bz * B - 1, 0)
        data[z0:bz * B + B + 1, y0:by * B + B + 1, x0:bx * B + B + 1] = faint[z0:bz * B + B + 1, y0:by * B + B + 1, x0:bx * B + B + 1]
    vol = oracle.Volume(nx, ny, nz, B, 1, data=data)
    tf = synth.tf_ramp()
    tf[:64, 3] = 0.0                                 # zero opacity below u = 0.25 (value 0.25)
    vol.set_transfer_function(tf, synth.TF_VMIN, synth.TF_VMAX)
    transparent = [b for b in range(vol.nbricks) if vol.brick_transparent(b)]
    assert transparent == [0, 5, 7]
    W, H = 48, 36
    fr = synth.Framing(nx, ny, nz, W, H)
    r = vol.render(fr.seeded(3, 1), fr.proj(False), W, H, 0.5, oracle.ALPHA, want_sub=True)
    sub = r["sub"].reshape(H * W, vol.nbricks, 4)
    assert np.all(sub[:, transparent, :] == 0.0)
    assert np.abs(sub[:, [b for b in range(vol.nbricks) if b not in transparent], 3]).max() > 0.1


# --------------------------------------------------------------------------- per-ray step (row f2 (i), R18)
def test_auto_step_is_one_sample_per_major_axis_voxel():
    """PAPER.md:152 "at least one sample for each voxel intersected": step = 0 selects
    1 / max|d_a| per ray. Closed forms: the number of scheduled samples is ceil(chord * max|d_a|)
    = the number of unit slabs crossed along the major axis; an axis-aligned view is the
    step-1 render; the homogeneous cube keeps its exact opacity (the weights sum to the chord)."""
    n = 24
    data = small_noise(n, n, n, seed=11)
    vol = oracle.Volume(n, n, n, 8, 1, data=data)
    vol.set_transfer_function(synth.tf_translucent(), -3, 10)
    vol.set_early_termination(2.0)
    W, H = 40, 30
    fr = synth.Framing(n, n, n, W, H)
    for ortho in (False, True):
        view, proj = fr.seeded(3, 1), fr.proj(ortho)
        r = vol.render(view, proj, W, H, 0.0, oracle.ALPHA)
        sched = r["counts"][..., 1]
        checked = 0
        for (i, j) in ((W // 2, H // 2), (W // 3, H // 2), (W // 2, H // 3), (2 * W // 3, 2 * H // 3), (5, 5)):
            o, d, tfar = ray_np(view, proj, W, H, i, j)
            c = chord_np(o, d, tfar, [n, n, n])
            if c is not None:
                t0, t1 = c
                expect = math.ceil((t1 - t0) * np.abs(d).max() - 1e-9)
                assert abs(int(sched[j, i]) - expect) <= 1 and sched[j, i] >= expect - 1e-9, (i, j, sched[j, i], expect)
                checked += 1
            else:
                assert sched[j, i] == 0
        assert checked >= 3
    view, proj = ortho_along_z(n, n, n)
    a = vol.render(view, proj, n, n, 0.0, oracle.ALPHA)["image"]
    b = vol.render(view, proj, n, n, 1.0, oracle.ALPHA)["image"]
    assert np.array_equal(a, b)
    # homogeneous cube: opacity 1 - (1 - a)^L whatever the step, so also with the per-ray step
    hom = oracle.Volume(n, n, n, 8, 1, data=np.full((n, n, n), 2.0, dtype=np.float32))
    hom.set_transfer_function(const_tf((0.2, 0.5, 0.9), 0.05), -3, 10)
    hom.set_early_termination(2.0)
    view, proj = fr.seeded(3, 2), fr.proj(False)
    img = hom.render(view, proj, W, H, 0.0, oracle.ALPHA)["image"]
    for (i, j) in ((W // 2, H // 2), (W // 3, H // 2), (W // 2, 2 * H // 3)):
        o, d, tfar = ray_np(view, proj, W, H, i, j)
        c = chord_np(o, d, tfar, [n, n, n])
        L = (c[1] - c[0]) if c is not None else 0.0
        a32 = float(np.float32(0.05))                # the table holds float32 opacities
        assert L > 5 and abs(img[j, i, 3] - (1.0 - (1.0 - a32) ** L)) < 1e-12


# --------------------------------------------------------------------------- blanked voxels (R14)
def test_nan_voxels_drop_the_samples_that_rest_on_them():
    """Radio cubes blank voxels with NaN. R14: a sample with more than 4e-6 of its tri-linear
    weight on NaN voxels is dropped; otherwise the NaN corners are left out and the others
    renormalised (so a NaN neighbour with weight 0 changes nothing - where the paper's per-ray
    step puts whole rays). Closed forms: homogeneous cube, axis-aligned orthographic rays, step 1.
    (i) rays through voxel centres, a blanked slab of T planes: exactly the T samples in the slab
    vanish, opacity = 1 - (1-a)^(n - T); (ii) rays at quarter-voxel offsets, a blanked plane
    x = m: the rays with |x - (m + 1/2)| < 1 lose every sample, the others none; (iii) MIP of a
    z-ramp with its brightest planes blanked is the brightest surviving plane; the data range
    ignores NaN; a fully blanked cube renders nothing."""
    n, T, z0 = 20, 4, 9
    view, proj = ortho_along_z(n, n, n)
    a32 = float(np.float32(0.05))
    data = np.full((n, n, n), 2.0, dtype=np.float32)
    data[z0:z0 + T] = np.nan
    vol = oracle.Volume(n, n, n, 8, 1, data=data)
    vol.set_transfer_function(const_tf((0.2, 0.5, 0.9), 0.05), -3, 10)
    vol.set_early_termination(2.0)
    r = vol.render(view, proj, n, n, 1.0, oracle.ALPHA)
    assert np.abs(r["image"][..., 3] - (1.0 - (1.0 - a32) ** (n - T))).max() < 1e-12
    assert np.all(r["counts"][..., 0] == n - T) and np.all(r["counts"][..., 1] == n)
    assert not (r["flags"] & oracle.FLAG_NAN_MARGIN).any()
    # (ii) a blanked plane x = m seen at two pixels per voxel
    m = 7
    data2 = np.full((n, n, n), 2.0, dtype=np.float32)
    data2[:, :, m] = np.nan
    vol2 = oracle.Volume(n, n, n, 8, 1, data=data2)
    vol2.set_transfer_function(const_tf((0.2, 0.5, 0.9), 0.05), -3, 10)
    vol2.set_early_termination(2.0)
    r2 = vol2.render(view, proj, 2 * n, n, 1.0, oracle.ALPHA)
    taken = r2["counts"][0, :, 0]
    xs = (np.arange(2 * n) + 0.5) / 2.0                       # pixel centres in voxel units (either orientation:
    hit = np.abs(xs - (m + 0.5)) < 1.0                        # the test cube is symmetric under x -> n - x only if
    hit_m = np.abs((n - xs) - (m + 0.5)) < 1.0                # mirrored, so accept the view's handedness)
    assert (np.array_equal(taken == 0, hit) or np.array_equal(taken == 0, hit_m)) and set(np.unique(taken)) == {0, n}
    full = 1.0 - (1.0 - a32) ** n
    assert np.abs(r2["image"][0, taken == n, 3] - full).max() < 1e-12 and not r2["image"][0, taken == 0].any()
    # (iii)
    ramp = np.broadcast_to(np.arange(n, dtype=np.float32)[:, None, None], (n, n, n)).copy()
    ramp[n - 3:] = np.nan
    volr = oracle.Volume(n, n, n, 8, 1, data=ramp)
    tf = synth.tf_ramp()
    volr.set_transfer_function(tf, 0.0, float(n))
    mimg = volr.render(view, proj, n, n, 1.0, oracle.MIP)["image"]
    assert np.abs(mimg[..., 0] - (n - 4) / float(n)).max() < 1e-6 and np.all(mimg[..., 3] == 1.0)
    assert volr.brick_minmax(-1) == (np.float32(0.0), np.float32(n - 4))
    blank = oracle.Volume(n, n, n, 8, 1, data=np.full((n, n, n), np.nan, dtype=np.float32))
    blank.set_transfer_function(tf, 0.0, 1.0)
    for mode in (oracle.ALPHA, oracle.MIP):
        assert not blank.render(view, proj, n, n, 1.0, mode)["image"].any()


# --------------------------------------------------------------------------- a2: rendering rectangles are TIGHT
def test_rendering_rectangle_closed_form_axis_aligned():
    """PAPER.md:150 (sec. 2.3.2), Fig. 4 :168: the rendering rectangle is the bounding box of the 8 projected vertices.
    For the axis-aligned orthographic camera a brick [lo,hi) projects onto a pixel box known in closed form
    (pixel i looks down x = nx - (i+1/2) nx/W, pixel j down y = (j+1/2) ny/H): the rectangle must EQUAL it, not
    merely contain it - a whole-viewport rectangle or one rounded a pixel too wide fails here."""
    nx, ny, nz, brick = 19, 11, 13, 5
    W, H = 58, 47  # no brick face projects onto a pixel boundary: 58/19 and 47/11 times 5, 10, 15 are not integers
    view, proj = ortho_along_z(nx, ny, nz)
    vol = oracle.Volume(nx, ny, nz, brick, 1)
    rects = vol.rects(view, proj, W, H)
    assert vol.nbricks == 4 * 3 * 3
    for b in range(vol.nbricks):
        bx, by = b % 4, (b // 4) % 3
        lo = (bx * brick, by * brick)
        hi = (min(lo[0] + brick, nx), min(lo[1] + brick, ny))
        ex0, ex1 = (nx - hi[0]) * W / nx, (nx - lo[0]) * W / nx  # the look-at basis mirrors x
        ey0, ey1 = lo[1] * H / ny, hi[1] * H / ny
        for e in (ex0, ex1, ey0, ey1):  # the closed form is robust: far from an integer, or exactly on the viewport edge
            assert e in (0.0, float(W), float(H)) or abs(e - round(e)) > 1e-3
        want = [math.floor(ex0), math.floor(ey0), math.ceil(ex1), math.ceil(ey1)]
        # a face exactly on the viewport edge may round a hair outside it before clipping: same box
        want = [max(want[0], 0), max(want[1], 0), min(want[2], W), min(want[3], H)]
        assert rects[b].tolist() == want, (b, rects[b].tolist(), want)
    # every pixel whose ray takes a sample in a brick lies in its rectangle AND the rectangle ends within one pixel
    # of the first / last such pixel on every side (the rectangle covers every pixel the projection TOUCHES, a ray
    # goes through a pixel's centre; a brick face parallel to the image plane has no sharp corner to miss)
    data = np.ones((nz, ny, nx), dtype=np.float32)
    vol = oracle.Volume(nx, ny, nz, brick, 1, data=data)
    vol.set_transfer_function(const_tf((1, 1, 1), 0.5), 0.0, 2.0)
    pix = np.array([(i, j) for j in range(H) for i in range(W)], dtype=np.int32)
    res = vol.render(view, proj, W, H, 1.0, oracle.MIP, pixels=pix, want_sub=True)
    for b in range(vol.nbricks):
        hit = res["sub"][:, b, 1].reshape(H, W) > 0
        js, is_ = np.nonzero(hit)
        x0, y0, x1, y1 = rects[b].tolist()
        assert x0 <= is_.min() <= x0 + 1 and y0 <= js.min() <= y0 + 1
        assert x1 - 1 <= is_.max() + 1 <= x1 and y1 - 1 <= js.max() + 1 <= y1


@pytest.mark.parametrize("ortho", [False, True])
def test_rendering_rectangle_is_the_bounding_box_of_the_projected_brick(ortho):
    """The same for seeded oblique views, against numpy's own matrices: a dense lattice of points on the brick's 12
    edges (the 8 vertices included) is projected with P @ V; the rectangle must equal floor(min) .. ceil(max) of
    the projected points, clipped to the viewport (tight AND conservative), also for bricks partly off screen."""
    nx, ny, nz, brick = 37, 29, 23, 8
    W, H = 203, 117
    fr = synth.Framing(nx, ny, nz, W, H)
    vol = oracle.Volume(nx, ny, nz, brick, 1)
    g = [(n + brick - 1) // brick for n in (nx, ny, nz)]
    t = np.linspace(0.0, 1.0, 33)
    checked = clipped = 0
    for k in range(6):
        view = fr.seeded(31, k)
        if ortho:
            proj = synth.orthographic(0.6 * fr.R * fr.aspect, 0.6 * fr.R, fr.near, fr.far)  # zoomed in: bricks leave the viewport
        else:
            proj = synth.perspective(25.0, fr.aspect, fr.near, fr.far)
        V, P = mats(view, proj)
        M = P @ V
        rects = vol.rects(view, proj, W, H)
        for b in range(vol.nbricks):
            bc = (b % g[0], (b // g[0]) % g[1], b // (g[0] * g[1]))
            lo = np.array([c * brick for c in bc], dtype=np.float64)
            hi = np.minimum(lo + brick, (nx, ny, nz))
            pts = []
            for a in range(3):  # 4 edges along each axis
                for u in (lo, hi):
                    for w in (lo, hi):
                        p = np.empty((len(t), 3))
                        p[:, a] = lo[a] + t * (hi[a] - lo[a])
                        p[:, (a + 1) % 3] = u[(a + 1) % 3]
                        p[:, (a + 2) % 3] = w[(a + 2) % 3]
                        pts.append(p)
            pts = np.concatenate(pts)
            clip = np.c_[pts, np.ones(len(pts))] @ M.T
            assert (clip[:, 3] > 0).all()  # the camera is outside the volume in these views
            px = (clip[:, 0] / clip[:, 3] + 1.0) * 0.5 * W
            py = (clip[:, 1] / clip[:, 3] + 1.0) * 0.5 * H
            ext = [px.min(), py.min(), px.max(), py.max()]
            if any(abs(e - round(e)) < 1e-7 for e in ext):
                continue  # a vertex on a pixel boundary: floor / ceil is a coin toss between two valid boxes
            want = [int(np.clip(math.floor(ext[0]), 0, W)), int(np.clip(math.floor(ext[1]), 0, H)),
                    int(np.clip(math.ceil(ext[2]), 0, W)), int(np.clip(math.ceil(ext[3]), 0, H))]
            assert rects[b].tolist() == want, (k, b, rects[b].tolist(), want)
            checked += 1
            clipped += want != [math.floor(ext[0]), math.floor(ext[1]), math.ceil(ext[2]), math.ceil(ext[3])]
    assert checked > 300 and clipped > 20


def test_rendering_rectangle_with_a_vertex_behind_the_eye_is_the_viewport():
    """a projected vertex is only meaningful in front of the eye; a brick with a vertex at clip w <= 0
    gets the whole viewport (conservative), bricks entirely in front keep tight boxes."""
    nx = ny = nz = 16
    vol = oracle.Volume(nx, ny, nz, 8, 1)
    W, H = 64, 48
    view = synth.look_at((8.0, 8.0, 6.0), (8.0, 8.0, 16.0), (0.0, 1.0, 0.0))  # inside, looking up +z
    proj = synth.perspective(60.0, W / H, 0.1, 100.0)
    rects = vol.rects(view, proj, W, H)
    for b in range(8):
        if b < 4:   # z in [0, 8): holds vertices behind the eye plane z = 6
            assert rects[b].tolist() == [0, 0, W, H]
        else:       # z in [8, 16]: in front; its far face is smaller than the viewport in one direction at least
            x0, y0, x1, y1 = rects[b]
            assert (x1 - x0) * (y1 - y0) < W * H


def test_margin_candidates_of_the_oracle():
    """R12 test hooks: on data without marginal decisions the candidate frames (tau -/+ 1e-5, NaN limit x0.5 / x2)
    equal the frame itself; with a blanked voxel and a sample whose NaN weight sits inside the flag's band the two
    limits give the dropped and the kept value, and the nominal limit gives one of them."""
    nx, ny, nz = 12, 10, 9
    data = small_noise(nx, ny, nz)
    W, H = 24, 20
    fr = synth.Framing(nx, ny, nz, W, H)
    view, proj = fr.seeded(2, 1), fr.proj(False)
    vol = oracle.Volume(nx, ny, nz, 5, 1, data=data)
    vol.set_transfer_function(synth.tf_translucent(), -3, 10)
    ref = vol.render(view, proj, W, H, 0.5, oracle.ALPHA)
    assert not ref["flags"].any() or not (ref["flags"] & (oracle.FLAG_ERT_MARGIN | oracle.FLAG_NAN_MARGIN)).any()
    for dtau, ns in ((-1e-5, 1.0), (1e-5, 1.0), (0.0, 0.5), (0.0, 2.0)):
        assert np.array_equal(ref["alt"](dtau, ns)["image"], ref["image"])
    assert np.array_equal(vol.render(view, proj, W, H, 0.5, oracle.ALPHA)["image"], ref["image"])  # the hooks were reset
    # one blanked voxel on the axis of an axis-aligned ray bundle; lateral offset chosen so that the NaN corner's
    # weight is 3e-6 (inside (2e-6, 8e-6)): dropped with the limit at 2e-6, kept and renormalised at 4e-6 and 8e-6
    n = 8
    d = np.full((n, n, n), 2.0, dtype=np.float32)
    d[:, 3, 3] = np.nan  # a blanked line of voxels along z at x = y = 3 (centres at 3.5)
    o = oracle.Volume(n, n, n, 8, 1, data=d)
    o.set_transfer_function(synth.tf_ramp(), 0.0, 4.0)
    eps = 3e-6
    view2 = synth.look_at((2.5 + eps, 2.5, -10.0), (2.5 + eps, 2.5, 0.0), (0.0, 1.0, 0.0))
    proj2 = synth.orthographic(1e-3, 1e-3, 1.0, 40.0)
    r = o.render(view2, proj2, 1, 1, 1.0, oracle.MIP)
    # pixel (0,0) looks down x = 2.5 + eps (mirrored basis: centre pixel = centre line), y = 2.5: weights on the
    # x = 3 column are eps, on y = 3 are 0, so the NaN corner (3,3) has weight 0 ... the ray is kept at any limit
    assert r["image"][0, 0, 3] == 1.0
    view3 = synth.look_at((3.0 - eps, 3.0 - 1e-9, -10.0), (3.0 - eps, 3.0 - 1e-9, 0.0), (0.0, 1.0, 0.0))
    r = o.render(view3, proj2, 1, 1, 1.0, oracle.MIP)
    # x = 3 - eps -> q_x = 2.5 - eps: cell 2, weight on column 3 = 0.5 - eps; y likewise ~0.5: N ~ 0.25: dropped at every limit
    assert r["image"][0, 0, 3] == 0.0
    # weight exactly in the band: sample at q = (2 + s, 2 + s) with s^2 = 3e-6
    s = math.sqrt(3e-6)
    view4 = synth.look_at((2.5 + s, 2.5 + s, -10.0), (2.5 + s, 2.5 + s, 0.0), (0.0, 1.0, 0.0))
    r = o.render(view4, proj2, 1, 1, 1.0, oracle.MIP)
    assert (r["flags"] & oracle.FLAG_NAN_MARGIN).all()
    kept, dropped = r["alt"](0.0, 2.0), r["alt"](0.0, 0.5)
    assert kept["image"][0, 0, 3] == 1.0 and kept["counts"][0, 0, 0] == n
    assert dropped["image"][0, 0, 3] == 0.0 and dropped["counts"][0, 0, 0] == 0
    assert np.array_equal(r["image"], kept["image"])  # 3e-6 < 4e-6: the nominal limit keeps it
