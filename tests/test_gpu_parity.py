"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle on the same seeded
inputs. Tolerances are north_star's: ALPHA max abs 2e-3 per RGBA channel, MIP 1e-5 relative;
brick order, rectangles and ray-brick lists exact; brick store bit-exact."""
import numpy as np
import pytest

import oracle
import synth
from helpers import check_alpha, check_mip, gpu_frame, make_pair, seeded_pixels

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def vr(cuda_device):
    from paper_1205_0282_b200 import build
    build.build()
    import paper_1205_0282_b200 as vr
    return vr


def views_for(cube, W, H, n_rot=3, seed=77):
    fr = synth.Framing(cube.nx, cube.ny, cube.nz, W, H)
    out = []
    for ortho in (False, True):
        for k in range(n_rot):
            out.append((("ortho" if ortho else "persp") + str(k), fr.seeded(seed, k), fr.proj(ortho)))
    return out


# --------------------------------------------------------------------------- inputs
@pytest.mark.parametrize("kind", [0, 1])
def test_device_generator_is_the_host_generator(vr, kind):
    """synth's CUDA twin makes bit-identical cubes (it is what fills the 103 GB store), both kinds."""
    import torch
    c = synth.Cube(77, 70, 45, 33, 9, ramp=0.5, kind=kind)
    dev = torch.empty((20, 30, 50), dtype=torch.float32, device="cuda")
    c.fill_device(dev.data_ptr(), 11, 7, 5, 50, 30, 20, torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    assert np.array_equal(dev.cpu().numpy(), c.fill_host(11, 7, 5, 50, 30, 20))


# --------------------------------------------------------------------------- a1 brick store
@pytest.mark.parametrize("ghost", [0, 1, 2])
def test_brick_store_is_bit_exact(vr, ghost):
    import torch
    cube = synth.Cube(5, 37, 29, 23, 3)
    data = cube.fill_host()
    g = vr.Volume(37, 29, 23, 8, ghost)
    o = oracle.Volume(37, 29, 23, 8, ghost, data=data)
    g.upload(data)  # host path
    for b in range(g.nbricks):
        assert np.array_equal(g.debug_brick_data(b), o.brick_data(b)), b
    back = np.zeros_like(data)
    g.download(back)
    assert np.array_equal(back, data)
    # device path, z-slabs and an interior sub-box written last
    g2 = vr.Volume(37, 29, 23, 8, ghost)
    d = torch.from_numpy(data).cuda()
    for z0 in range(0, 23, 5):
        g2.upload(d[z0:z0 + 5].contiguous(), origin=(0, 0, z0))
    g2.upload(d[3:9, 4:20, 6:30].contiguous(), origin=(6, 4, 3))
    for b in range(g2.nbricks):
        assert np.array_equal(g2.debug_brick_data(b), o.brick_data(b)), b
    sub = torch.zeros((7, 9, 11), dtype=torch.float32, device="cuda")
    g2.download(sub, origin=(13, 10, 8))
    assert np.array_equal(sub.cpu().numpy(), data[8:15, 10:19, 13:24])


def test_tma_upload_path_gives_the_same_store(vr):
    """vr_debug_set_upload_path: the TMA box-load kernel (cp.async.bulk.tensor, the default) and the cp.async staging kernel
    (its fallback) fill the store identically, ragged bricks, volume faces (edge replication), sub-box uploads and boxes
    the tensor map cannot describe (a row length that is not a multiple of 4 cells) included."""
    import torch
    for dims, brick, ghost in (((128, 96, 80), 32, 1), ((100, 72, 50), 32, 2), ((64, 64, 64), 64, 1), ((101, 72, 50), 32, 1)):
        data = synth.Cube(6, *dims, 3).fill_host()
        o = oracle.Volume(*dims, brick, ghost, data=data)
        d = torch.from_numpy(data).cuda()
        try:
            for path in (1, 0):
                vr.debug_set_upload_path(path)
                g = vr.Volume(*dims, brick, ghost)
                for z0 in range(0, dims[2], 24):                   # z-slabs, then interior sub-boxes written again
                    g.upload(d[z0:z0 + 24].contiguous(), origin=(0, 0, z0))
                g.upload(d[8:40, 12:60, 20:84].contiguous(), origin=(20, 12, 8))
                g.upload(d[3:30, 5:41, 7:70].contiguous(), origin=(7, 5, 3))     # 63 cells per row: the cp.async kernel either way
                for b in range(g.nbricks):
                    assert np.array_equal(g.debug_brick_data(b), o.brick_data(b)), (dims, b, path)
                g.close()
        finally:
            vr.debug_set_upload_path(1)


@pytest.mark.parametrize("case", range(int(__import__("os").environ.get("VR_UPLOAD_CASES", "24"))))
def test_randomised_uploads(vr, case):
    """Row a1 under random use: volumes with ragged bricks, ghost 0-2, bricks of 8-256 cells (rows of one to three 128-cell
    chunks plus tails), a whole-volume upload followed by random sub-boxes of new data (row lengths and origins that the
    tensor map can and cannot describe, device and host sources): every brick equals the oracle's copy of the final volume,
    and the volume comes back unchanged."""
    import torch
    rng = np.random.default_rng(9000 + case)
    brick = int(rng.choice([8, 16, 32, 64, 128, 256]))
    dims = tuple(int(v) for v in rng.integers(max(9, brick // 2), min(300, 3 * brick + 40), 3))
    if brick >= 128:  # keep the oracle's copies small: one long axis is enough to cross chunk boundaries
        dims = (int(rng.integers(130, 420)), int(rng.integers(20, 70)), int(rng.integers(10, 40)))
    ghost = int(rng.choice([0, 1, 1, 2]))
    nx, ny, nz = dims
    data = rng.standard_normal((nz, ny, nx)).astype(np.float32)
    g = vr.Volume(nx, ny, nz, brick, ghost)
    g.upload(torch.from_numpy(data).cuda() if case % 2 else data)
    for k in range(int(rng.integers(1, 5))):
        sx, sy, sz = (int(rng.integers(1, d + 1)) for d in dims)
        if rng.random() < 0.5:
            sx = max(4, sx & ~3)                      # a row length the tensor map can describe
        sx = min(sx, nx)
        x0, y0, z0 = int(rng.integers(0, nx - sx + 1)), int(rng.integers(0, ny - sy + 1)), int(rng.integers(0, nz - sz + 1))
        patch = rng.standard_normal((sz, sy, sx)).astype(np.float32)
        if rng.random() < 0.3:
            patch[rng.random(patch.shape) < 0.02] = np.nan   # blanked voxels (R14)
        data[z0:z0 + sz, y0:y0 + sy, x0:x0 + sx] = patch
        g.upload(torch.from_numpy(patch).cuda() if (case + k) % 3 else patch, origin=(x0, y0, z0))
    o = oracle.Volume(nx, ny, nz, brick, ghost, data=data)
    for b in range(g.nbricks):
        assert np.array_equal(g.debug_brick_data(b), o.brick_data(b), equal_nan=True), (case, dims, brick, ghost, b)
    # row f1 after the last upload: the per-brick ranges (one streaming read, integer atomics) equal the oracle's, blanked voxels ignored
    mm = g.debug_brick_minmax()
    for b in range(g.nbricks):
        assert tuple(mm[b]) == o.brick_minmax(b), (case, b)
    back = np.zeros_like(data)
    g.download(back)
    assert np.array_equal(back, data, equal_nan=True)
    g.close()


# --------------------------------------------------------------------------- a2, a3
@pytest.mark.parametrize("dims,brick", [((64, 64, 64), 64), ((100, 90, 70), 32), ((37, 29, 23), 8)])
def test_brick_order_and_rectangles_match_exactly(vr, dims, brick):
    nx, ny, nz = dims
    g = vr.Volume(nx, ny, nz, brick, 1)
    o = oracle.Volume(nx, ny, nz, brick, 1)
    W, H = 203, 117
    fr = synth.Framing(nx, ny, nz, W, H)
    cases = [(fr.seeded(3, k), fr.proj(k % 2 == 1)) for k in range(12)]
    cases += [(fr.turntable(k), fr.proj(False)) for k in range(0, 36, 5)]
    # eye inside the volume / close to a face: slabs at distance 0
    cases.append((synth.look_at((nx * 0.4, ny * 0.6, nz * 0.5), (nx, ny, nz), (0, 0, 1)), synth.perspective(60, W / H, 0.5, 500)))
    for view, proj in cases:
        assert np.array_equal(g.debug_brick_order(view, proj), o.brick_order(view, proj))
        assert np.array_equal(g.debug_rects(view, proj, W, H), o.rects(view, proj, W, H))


def test_ray_brick_lists_match_exactly(vr):
    nx, ny, nz, brick = 100, 90, 70, 32
    g = vr.Volume(nx, ny, nz, brick, 1)
    o = oracle.Volume(nx, ny, nz, brick, 1)
    W, H = 160, 120
    fr = synth.Framing(nx, ny, nz, W, H)
    pix = seeded_pixels(9, W, H, 4000)
    for k in range(6):
        view, proj = fr.seeded(5, k), fr.proj(k % 2 == 1)
        gc, gl, gg = g.debug_ray_bricks(view, proj, W, H, pix, maxlen=16)
        oc, ol, og = o.ray_bricks(view, proj, W, H, pix, maxlen=16)
        ok = (gg == 0) & (og == 0)
        assert ok.mean() > 0.99
        assert np.array_equal(gc[ok], oc[ok])
        assert np.array_equal(gl[ok], ol[ok])
        assert oc.max() > 3  # the lists are not trivial


# --------------------------------------------------------------------------- c0: one brick
@pytest.mark.parametrize("tf_name", ["ramp", "translucent"])
def test_config0_full_frames(vr, tf_name):
    c = synth.CONFIGS["c0"]
    cube = synth.config_cube("c0")
    tf = synth.tf_ramp() if tf_name == "ramp" else synth.tf_translucent()
    g, o = make_pair(cube, c["brick"], c["ghost"], tf=tf)
    W, H = c["width"], c["height"]
    for name, view, proj in views_for(cube, W, H):
        ref = o.render(view, proj, W, H, c["step"], oracle.ALPHA)
        check_alpha(gpu_frame(g, view, proj, W, H, c["step"], vr.ALPHA), ref, 0.99, "c0 " + name)
        ref = o.render(view, proj, W, H, c["step"], oracle.MIP)
        check_mip(gpu_frame(g, view, proj, W, H, c["step"], vr.MIP), ref, "c0 " + name)
        assert ref["image"][..., 3].max() == 1.0 and ref["image"][..., 3].min() == 0.0


# --------------------------------------------------------------------------- bricked, ragged
@pytest.mark.parametrize("tau", [0.99, 2.0])
def test_bricked_ragged_full_frames_and_subimages(vr, tau):
    cube = synth.Cube(11, 100, 90, 70, 12)
    tf = synth.tf_translucent() if tau > 1 else synth.tf_ramp()
    g, o = make_pair(cube, 32, 1, tf=tf, tau=tau)
    W, H = 203, 117  # not multiples of the 8x4 tile
    step = 0.5
    pix = seeded_pixels(4, W, H, 300)
    for name, view, proj in views_for(cube, W, H, n_rot=2):
        ref = o.render(view, proj, W, H, step, oracle.ALPHA)
        img = gpu_frame(g, view, proj, W, H, step, vr.ALPHA)
        check_alpha(img, ref, tau, name)
        # row a8: each brick's sub-image value
        sub_ref = o.render(view, proj, W, H, step, oracle.ALPHA, pixels=pix, want_sub=True)
        sub = g.debug_subimages(pix).astype(np.float64)
        check_alpha(sub, sub_ref, tau, name + " sub-images", key="sub")
        ref = o.render(view, proj, W, H, step, oracle.MIP)
        check_mip(gpu_frame(g, view, proj, W, H, step, vr.MIP), ref, name)
        sub_ref = o.render(view, proj, W, H, step, oracle.MIP, pixels=pix, want_sub=True)
        sub = g.debug_subimages(pix).astype(np.float64)[..., 0]
        m_ref = sub_ref["sub"][..., 0]
        assert np.array_equal(np.isinf(sub), np.isinf(m_ref))  # same bricks took samples
        fin = ~np.isinf(m_ref)
        # the kernel may stop a MIP ray once the running max reaches vmax
        check_mip(np.minimum(sub[fin], synth.TF_VMAX), np.minimum(m_ref[fin], synth.TF_VMAX), name + " sub-image max")


def test_one_brick_equals_n_bricks_on_gpu(vr):
    """ERT off: the bricked result equals the single-brick result (ghost = 1 suffices, R3)."""
    cube = synth.Cube(12, 60, 50, 40, 5)
    data = cube.fill_host()
    tf = synth.tf_translucent()
    g1, _ = make_pair(cube, 64, 1, tf=tf, tau=2.0, data=data)
    gn, _ = make_pair(cube, 16, 1, tf=tf, tau=2.0, data=data)
    g0, _ = make_pair(cube, 16, 0, tf=tf, tau=2.0, data=data)
    W, H = 128, 96
    fr = synth.Framing(60, 50, 40, W, H)
    view, proj = fr.seeded(2, 0), fr.proj(False)
    a = gpu_frame(g1, view, proj, W, H, 0.5, vr.ALPHA)
    b = gpu_frame(gn, view, proj, W, H, 0.5, vr.ALPHA)
    c = gpu_frame(g0, view, proj, W, H, 0.5, vr.ALPHA)
    assert np.abs(a - b).max() < 2e-5
    assert np.abs(a - c).max() > 1e-3  # ghost = 0 must show seams (negative test)
    am = gpu_frame(g1, view, proj, W, H, 0.5, vr.MIP)
    bm = gpu_frame(gn, view, proj, W, H, 0.5, vr.MIP)
    check_mip(bm, am, "1 vs N bricks")


def test_pipelined_host_frames_equal_synchronous_ones(vr):
    """vr_render_host_async / vr_render_host_wait: six frames in flight two at a time arrive
    bit-identical to vr_render_host's, and the first one matches the oracle."""
    import torch
    cube = synth.Cube(21, 72, 40, 56, 6)
    g, o = make_pair(cube, 32, 1)
    W, H = 144, 100
    fr = synth.Framing(cube.nx, cube.ny, cube.nz, W, H)
    views = [fr.turntable(k) for k in range(6)]
    proj = fr.proj(False)
    bufs = [torch.empty((H, W, 4), dtype=torch.float32).pin_memory() for _ in views]
    for mode in (vr.ALPHA, vr.MIP):
        for b in bufs:
            b.fill_(-1.0)
        for v, b in zip(views, bufs):
            g.render_host_async(v, proj, W, H, 0.5, mode, b)
        g.render_host_wait()
        for v, b in zip(views, bufs):
            sync = g.render_host(v, proj, W, H, 0.5, mode)
            assert np.array_equal(b.numpy(), sync)
    ref = o.render(views[0], proj, W, H, 0.5, oracle.MIP)
    check_mip(bufs[0].numpy().astype(np.float64), ref, "pipelined frame 0")


def test_host_entries_mixed_at_growing_sizes(vr):
    """The synchronous and the pipelined host entry own separate device frames: growing the frame of one
    must leave the other's frames, events and copy stream alone (small sync, async, LARGER sync, async, destroy)."""
    import torch
    cube = synth.Cube(22, 48, 40, 36, 4)
    g, o = make_pair(cube, 32, 1)
    small, large = (96, 64), (160, 120)
    frs = {s: synth.Framing(cube.nx, cube.ny, cube.nz, *s) for s in (small, large)}

    def sync(size, k):
        fr = frs[size]
        return g.render_host(fr.turntable(k), fr.proj(False), size[0], size[1], 0.5, vr.ALPHA)

    def pipelined(size, k):
        fr = frs[size]
        b = torch.full((size[1], size[0], 4), -1.0, dtype=torch.float32).pin_memory()
        g.render_host_async(fr.turntable(k), fr.proj(False), size[0], size[1], 0.5, vr.ALPHA, b)
        g.render_host_wait()
        return b.numpy().copy()

    a0 = sync(small, 1)
    assert np.array_equal(pipelined(small, 1), a0)
    a1 = sync(large, 2)                       # grows the synchronous frame only
    assert np.array_equal(pipelined(small, 1), a0)   # the pipelined frames, events and stream are still alive
    assert np.array_equal(pipelined(large, 2), a1)   # and can grow on their own
    assert np.array_equal(sync(small, 1), a0)
    ref = o.render(frs[large].turntable(2), frs[large].proj(False), large[0], large[1], 0.5, oracle.ALPHA)
    check_alpha(a1.astype(np.float64), ref, 0.99, "mixed host entries")
    g.close()


# --------------------------------------------------------------------------- f2 (i) per-ray step (R18)
@pytest.mark.parametrize("ortho", [False, True])
def test_auto_step_matches_oracle(vr, ortho):
    """step = VR_STEP_AUTO: 1 / max|d_a| per ray, sort-last and fused, ALPHA and MIP,
    with the exact sample count of the oracle."""
    cube = synth.Cube(61, 66, 50, 41, 5)
    data = cube.fill_host()
    g, o = make_pair(cube, 16, 1, data=data)
    one = oracle.Volume(cube.nx, cube.ny, cube.nz, 128, 1, data=data)
    one.set_transfer_function(synth.tf_ramp(), synth.TF_VMIN, synth.TF_VMAX)
    W, H = 150, 110
    fr = synth.Framing(cube.nx, cube.ny, cube.nz, W, H)
    view, proj = fr.seeded(6, 0), fr.proj(ortho)
    g.set_counting(1)
    for trav, orc in ((vr.SORT_LAST, o), (vr.FUSED, one)):
        g.set_traversal(trav)
        ref = orc.render(view, proj, W, H, 0.0, oracle.ALPHA)
        check_alpha(gpu_frame(g, view, proj, W, H, vr.STEP_AUTO, vr.ALPHA), ref, 0.99, "auto step")
        assert g.debug_stats()["samples"] == int(ref["counts"][..., 0].sum())
        check_mip(gpu_frame(g, view, proj, W, H, vr.STEP_AUTO, vr.MIP), orc.render(view, proj, W, H, 0.0, oracle.MIP), "auto step")
    # axis-aligned orthographic view: the per-ray step is exactly 1
    g.set_traversal(vr.SORT_LAST)
    view = synth.look_at((33, 25, -10.0), (33, 25, 0.0), (0.0, 1.0, 0.0))
    proj = synth.orthographic(33, 25, 1.0, 70.0)
    assert np.array_equal(gpu_frame(g, view, proj, 66, 50, vr.STEP_AUTO, vr.ALPHA), gpu_frame(g, view, proj, 66, 50, 1.0, vr.ALPHA))


# --------------------------------------------------------------------------- other bricks, ghosts, layouts
@pytest.mark.parametrize("brick,ghost,tile", [(20, 1, None), (7, 2, None), (24, 1, "3,1,1,0,0,0"), (20, 2, "1,2,2,1,1,1"),
                                               (12, 1, "linear")])
def test_odd_bricks_ghosts_and_generic_layouts(vr, monkeypatch, brick, ghost, tile):
    """Bricks that are not powers of two (the owner rule divides instead of scaling), wider ghost
    layers, x-linear rows and the generic separable micro-tile layouts (8x2x2 tiles; 2x4x4 tiles
    in 2x2x2 macro blocks) all render the same frames: parity with the oracle in both modes and
    both traversals, brick store and data range bit-exact."""
    cube = synth.Cube(57, 61, 47, 39, 5)
    data = cube.fill_host()
    layout = vr.LAYOUT_DEFAULT
    if tile == "linear":
        layout = vr.LAYOUT_LINEAR
    elif tile:
        monkeypatch.setenv("VR_TILE", tile)
    g = vr.Volume(61, 47, 39, brick, ghost, layout=layout)
    monkeypatch.delenv("VR_TILE", raising=False)
    g.upload(data)
    o = oracle.Volume(61, 47, 39, brick, ghost, data=data)
    one = oracle.Volume(61, 47, 39, 64, 1, data=data)
    for v in (g, o, one):
        v.set_transfer_function(synth.tf_ramp(), synth.TF_VMIN, synth.TF_VMAX)
        v.set_early_termination(0.99)
    back = np.empty_like(data)
    g.download(back)
    assert np.array_equal(back, data)
    for b in (0, g.nbricks // 2, g.nbricks - 1):
        assert np.array_equal(g.debug_brick_data(b), o.brick_data(b))
        assert tuple(g.debug_brick_minmax()[b]) == o.brick_minmax(b)
    W, H = 120, 90
    fr = synth.Framing(61, 47, 39, W, H)
    view, proj = fr.seeded(4, 2), fr.proj(False)
    assert np.array_equal(g.debug_brick_order(view, proj), o.brick_order(view, proj))
    ref = o.render(view, proj, W, H, 0.5, oracle.ALPHA)
    check_alpha(gpu_frame(g, view, proj, W, H, 0.5, vr.ALPHA), ref, 0.99, "sort-last")
    check_mip(gpu_frame(g, view, proj, W, H, 0.5, vr.MIP), o.render(view, proj, W, H, 0.5, oracle.MIP), "sort-last")
    g.set_traversal(vr.FUSED)
    ref = one.render(view, proj, W, H, 0.5, oracle.ALPHA)
    check_alpha(gpu_frame(g, view, proj, W, H, 0.5, vr.ALPHA), ref, 0.99, "fused")
    check_mip(gpu_frame(g, view, proj, W, H, 0.5, vr.MIP), one.render(view, proj, W, H, 0.5, oracle.MIP), "fused")


# --------------------------------------------------------------------------- f1 data range, culling
@pytest.mark.parametrize("layout", ["tiled", "linear"])
@pytest.mark.parametrize("ghost", [0, 1, 2])
def test_brick_minmax_is_exact(vr, layout, ghost):
    """Per-brick and global data range on a ragged grid: bit-equal to the oracle's."""
    cube = synth.Cube(41, 45, 38, 27, 4)
    data = cube.fill_host()
    lay = vr.LAYOUT_TILED if layout == "tiled" else vr.LAYOUT_LINEAR
    g = vr.Volume(45, 38, 27, 16, ghost, layout=lay)
    g.upload(data)
    o = oracle.Volume(45, 38, 27, 16, ghost, data=data)
    mm = g.debug_brick_minmax()
    for b in range(g.nbricks):
        assert tuple(mm[b]) == o.brick_minmax(b), b
    assert g.minmax() == o.brick_minmax(-1) == (data.min(), data.max())
    # a second upload invalidates the table: overwrite one voxel with a new maximum
    spike = np.full((1, 1, 1), 99.0, dtype=np.float32)
    g.upload(spike, origin=(44, 37, 26))
    assert g.minmax() == (data.min(), np.float32(99.0))


def sparse_cube(nx, ny, nz, B, seed):
    """N-body-like stand-in (Table 1 :221, the paper's other data family): most bricks hold
    only faint values (below the opacity threshold of the test's transfer function), a few hold
    the usual noise + sources."""
    data = synth.Cube(seed, nx, ny, nz, 6).fill_host()
    faint = np.clip(data, -2.9, -1.2)
    gx, gy, gz = -(-nx // B), -(-ny // B), -(-nz // B)
    for bz in range(gz):
        for by in range(gy):
            for bx in range(gx):
                if synth.u01(seed, 91, (bz * gy + by) * gx + bx) < 0.6:
                    x0, y0, z0 = max(bx * B - 1, 0), max(by * B - 1, 0), max(bz * B - 1, 0)
                    sl = (slice(z0, bz * B + B + 1), slice(y0, by * B + B + 1), slice(x0, bx * B + B + 1))
                    data[sl] = faint[sl]
    return data


def test_transparent_bricks_are_culled_exactly(vr):
    """R16: the set of culled bricks equals the oracle's transparent set, the frame still matches
    the oracle, and it is bit-identical with culling switched off."""
    import torch
    nx, ny, nz, B = 96, 72, 64, 16
    data = sparse_cube(nx, ny, nz, B, 17)
    tf = synth.tf_ramp()
    tf[:64, 3] = 0.0
    g = vr.Volume(nx, ny, nz, B, 1)
    g.upload(data)
    o = oracle.Volume(nx, ny, nz, B, 1, data=data)
    for v in (g, o):
        v.set_transfer_function(tf, synth.TF_VMIN, synth.TF_VMAX)
        v.set_early_termination(0.99)
    transparent = [b for b in range(o.nbricks) if o.brick_transparent(b)]
    assert 10 < len(transparent) < o.nbricks - 10
    W, H = 200, 150
    fr = synth.Framing(nx, ny, nz, W, H)
    view, proj = fr.seeded(8, 2), fr.proj(False)
    on = gpu_frame(g, view, proj, W, H, 0.5, vr.ALPHA)
    st = g.debug_stats()
    rects = o.rects(view, proj, W, H)
    visible = [b for b in transparent if rects[b][2] > rects[b][0] and rects[b][3] > rects[b][1]]
    assert st["bricks_culled"] == len(visible)
    pix = seeded_pixels(3, W, H, 64)
    subs = g.debug_subimages(pix)                    # [npix][nbricks][4]: culled bricks deliver nothing
    assert np.all(subs[:, transparent, :] == 0.0)
    ref = o.render(view, proj, W, H, 0.5, oracle.ALPHA)
    check_alpha(on, ref, 0.99, "culled frame")
    g.set_culling(False)
    off = gpu_frame(g, view, proj, W, H, 0.5, vr.ALPHA)
    assert g.debug_stats()["bricks_culled"] == 0
    assert np.array_equal(on, off)
    # the fused traversal skips the same bricks along each ray: same frame as with culling off, fewer samples
    one = oracle.Volume(nx, ny, nz, 128, 1, data=data)
    one.set_transfer_function(tf, synth.TF_VMIN, synth.TF_VMAX)
    g.set_traversal(vr.FUSED)
    g.set_counting(1)
    f_off = gpu_frame(g, view, proj, W, H, 0.5, vr.ALPHA)
    n_off = g.debug_stats()["samples"]
    g.set_culling(True)
    f_on = gpu_frame(g, view, proj, W, H, 0.5, vr.ALPHA)
    n_on = g.debug_stats()["samples"]
    assert np.array_equal(f_on, f_off) and n_on < 0.8 * n_off
    r1 = one.render(view, proj, W, H, 0.5, oracle.ALPHA)
    check_alpha(f_on, r1, 0.99, "fused, culled")
    g.set_counting(0)
    g.set_traversal(vr.SORT_LAST)
    g.set_culling(False)
    # MIP never culls, and stops at the global maximum of the data without changing the frame
    g.set_culling(True)
    m_on = gpu_frame(g, view, proj, W, H, 0.5, vr.MIP)
    assert g.debug_stats()["bricks_culled"] == 0
    g.set_culling(False)
    m_off = gpu_frame(g, view, proj, W, H, 0.5, vr.MIP)
    assert np.array_equal(m_on, m_off)
    check_mip(m_on, o.render(view, proj, W, H, 0.5, oracle.MIP), "MIP with data-max stop")


# --------------------------------------------------------------------------- R19 macro-cell skipping
def test_macro_cell_skipping_is_exact(vr):
    """A transfer function that hides the noise (alpha 0 below ~3.5 sigma, the usual way to look
    at a spectral cube): the 8x8x8 macro-cell flags equal an independent numpy statement of R19,
    frames are bit-identical with skipping on and off in both traversals, match the oracle, and
    most samples are never fetched."""
    nx, ny, nz, B = 100, 84, 60, 32                  # ragged 4 x 3 x 2 bricks
    cube = synth.Cube(71, nx, ny, nz, 10)
    data = cube.fill_host()
    tf = synth.tf_ramp()
    tf[:128, 3] = 0.0                                # opacity only above u = 0.5 (value 3.5)
    g = vr.Volume(nx, ny, nz, B, 1)
    g.upload(data)
    o = oracle.Volume(nx, ny, nz, B, 1, data=data)
    one = oracle.Volume(nx, ny, nz, 128, 1, data=data)
    for v in (g, o, one):
        v.set_transfer_function(tf, synth.TF_VMIN, synth.TF_VMAX)
        v.set_early_termination(0.99)
    # flags: numpy on the oracle's padded copy of the brick (float32 arithmetic of R16's entry rule)
    n = tf.shape[0]
    inv = np.float32(1.0 / (np.float64(np.float32(synth.TF_VMAX)) - np.float64(np.float32(synth.TF_VMIN))))

    def entry(x):
        u = np.clip((np.float32(x) - np.float32(synth.TF_VMIN)) * inv, np.float32(0), np.float32(1))
        return min(int(np.float32(u) * np.float32(n - 1)), n - 2)

    for b in (0, 5, g.nbricks - 1):
        pad = o.brick_data(b)                        # [dz][dy][dx] ghost-padded
        flags = g.debug_cell_flags(b)
        ncz, ncy, ncx = flags.shape
        seen = 0
        for mz in range(ncz):
            for my in range(ncy):
                for mx in range(ncx):
                    blk = pad[8 * mz:8 * mz + 9, 8 * my:8 * my + 9, 8 * mx:8 * mx + 9]   # the macro-cell + one layer
                    if blk.size == 0:
                        continue
                    i0, i1 = max(entry(blk.min()) - 1, 0), min(entry(blk.max()) + 2, n - 1)
                    assert flags[mz, my, mx] == int(not tf[i0:i1 + 1, 3].any()), (b, mx, my, mz)
                    seen += 1
        assert seen >= 8 and 0 < flags.sum()
    W, H = 200, 150
    fr = synth.Framing(nx, ny, nz, W, H)
    view, proj = fr.seeded(2, 1), fr.proj(False)
    g.set_counting(1)
    for trav, orc in ((vr.SORT_LAST, o), (vr.FUSED, one)):
        g.set_traversal(trav)
        g.set_culling(True)
        on = gpu_frame(g, view, proj, W, H, 0.5, vr.ALPHA)
        n_on = g.debug_stats()["samples"]
        g.set_culling(False)
        off = gpu_frame(g, view, proj, W, H, 0.5, vr.ALPHA)
        n_off = g.debug_stats()["samples"]
        assert np.array_equal(on, off) and on[..., 3].max() > 0.2
        assert n_on < 0.5 * n_off
        ref = orc.render(view, proj, W, H, 0.5, oracle.ALPHA)
        check_alpha(on, ref, 0.99, "macro-cell skipping")
        assert n_off == int(ref["counts"][..., 0].sum())
    # a new transfer function re-flags the cells; one without transparent entries switches skipping off
    g.set_traversal(vr.SORT_LAST)
    g.set_culling(True)
    g.set_transfer_function(synth.tf_ramp(), synth.TF_VMIN, synth.TF_VMAX)
    o.set_transfer_function(synth.tf_ramp(), synth.TF_VMIN, synth.TF_VMAX)
    ref = o.render(view, proj, W, H, 0.5, oracle.ALPHA)
    check_alpha(gpu_frame(g, view, proj, W, H, 0.5, vr.ALPHA), ref, 0.99, "ramp after threshold")
    # nothing is skipped any more (a termination decided in float32 may differ by one sample on a few rays, R12)
    assert abs(g.debug_stats()["samples"] - int(ref["counts"][..., 0].sum())) <= 1e-4 * ref["counts"][..., 0].sum()


def test_mip_steps_over_empty_space_exactly(vr):
    """R19 for MIP (the paper's shipped mode) on a density cube with a zero background: macro-cells
    that cannot raise a ray's maximum are stepped over; frames bit-identical with the feature off,
    equal to the oracle's, far fewer samples, in both traversals."""
    nx, ny, nz, B = 128, 96, 80, 32
    cube = synth.Cube(33, nx, ny, nz, 3, kind=synth.NBODY)
    data = cube.fill_host()
    assert (data == 0.0).mean() > 0.3
    tf = synth.tf_density()
    g = vr.Volume(nx, ny, nz, B, 1)
    g.upload(data)
    o = oracle.Volume(nx, ny, nz, B, 1, data=data)
    for v in (g, o):
        v.set_transfer_function(tf, 0.0, synth.NBODY_VMAX)
    W, H = 192, 144
    fr = synth.Framing(nx, ny, nz, W, H)
    view, proj = fr.seeded(9, 0), fr.proj(False)
    ref = o.render(view, proj, W, H, 0.5, oracle.MIP)
    g.set_counting(1)
    for trav in (vr.SORT_LAST, vr.FUSED):
        g.set_traversal(trav)
        g.set_culling(True)
        on = gpu_frame(g, view, proj, W, H, 0.5, vr.MIP)
        n_on = g.debug_stats()["samples"]
        g.set_culling(False)
        off = gpu_frame(g, view, proj, W, H, 0.5, vr.MIP)
        n_off = g.debug_stats()["samples"]
        assert np.array_equal(on, off) and n_on < 0.6 * n_off
        assert n_off == int(ref["counts"][..., 0].sum())
        check_mip(on, ref, "MIP over empty space")
    # a noise cube has no empty space: the feature stays off and every sample is taken
    noise = synth.Cube(34, 64, 48, 40, 2)
    gn, on_ = make_pair(noise, 16, 1)
    gn.set_counting(1)
    r2 = on_.render(view, proj, 64, 48, 0.5, oracle.MIP)
    fr2 = synth.Framing(64, 48, 40, 64, 48)
    r2 = on_.render(fr2.seeded(1, 0), fr2.proj(False), 64, 48, 0.5, oracle.MIP)
    check_mip(gpu_frame(gn, fr2.seeded(1, 0), fr2.proj(False), 64, 48, 0.5, vr.MIP), r2, "noise MIP")
    assert gn.debug_stats()["samples"] == int(r2["counts"][..., 0].sum())


# --------------------------------------------------------------------------- f2 fused traversal (R17)
@pytest.mark.parametrize("tau", [0.99, 2.0])
@pytest.mark.parametrize("ortho", [False, True])
def test_fused_traversal_equals_single_brick_oracle(vr, tau, ortho):
    """VR_FUSED on a ragged grid of bricks == the oracle holding the volume in ONE brick (R17):
    same sample schedule, global early termination. Also: the same frame on both layouts, and
    within rounding of the sort-last frame when early termination is off."""
    cube = synth.Cube(23, 70, 52, 44, 6)
    data = cube.fill_host()
    tf = synth.tf_ramp() if tau < 1 else synth.tf_translucent()
    g, _ = make_pair(cube, 16, 1, tf=tf, tau=tau, data=data)          # 5 x 4 x 3 bricks, ragged
    one = oracle.Volume(cube.nx, cube.ny, cube.nz, 128, 1, data=data)  # a single brick
    one.set_transfer_function(tf, synth.TF_VMIN, synth.TF_VMAX)
    one.set_early_termination(tau)
    W, H = 176, 132
    fr = synth.Framing(cube.nx, cube.ny, cube.nz, W, H)
    view, proj = fr.seeded(5, 1), fr.proj(ortho)
    g.set_traversal(vr.FUSED)
    g.minmax()                                                         # the once-per-upload range pass (f1)
    l0 = g.launch_count()
    fa = gpu_frame(g, view, proj, W, H, 0.5, vr.ALPHA)
    assert g.launch_count() - l0 == 2                                  # set-up + one fused kernel, no compositing
    ref = one.render(view, proj, W, H, 0.5, oracle.ALPHA)
    check_alpha(fa, ref, tau, "fused alpha")
    fm = gpu_frame(g, view, proj, W, H, 0.5, vr.MIP)
    check_mip(fm, one.render(view, proj, W, H, 0.5, oracle.MIP), "fused mip")
    g.set_traversal(vr.SORT_LAST)
    sm = gpu_frame(g, view, proj, W, H, 0.5, vr.MIP)
    check_mip(fm, sm, "fused vs sort-last mip")
    if tau > 1:
        sa = gpu_frame(g, view, proj, W, H, 0.5, vr.ALPHA)
        assert np.abs(sa - fa).max() < 2e-5
    # sample count: global termination takes no more samples than brick-local termination
    g.set_counting(1)
    gpu_frame(g, view, proj, W, H, 0.5, vr.ALPHA)
    n_sort = g.debug_stats()["samples"]
    g.set_traversal(vr.FUSED)
    gpu_frame(g, view, proj, W, H, 0.5, vr.ALPHA)
    n_fused = g.debug_stats()["samples"]
    assert n_fused == int(ref["counts"][..., 0].sum())                 # exactly the oracle's sample set
    assert n_fused <= n_sort
    g.set_counting(0)
    lin = vr.Volume(cube.nx, cube.ny, cube.nz, 16, 1, layout=vr.LAYOUT_LINEAR)
    lin.upload(data)
    lin.set_transfer_function(tf, synth.TF_VMIN, synth.TF_VMAX)
    lin.set_early_termination(tau)
    lin.set_traversal(vr.FUSED)
    assert np.array_equal(gpu_frame(lin, view, proj, W, H, 0.5, vr.ALPHA), fa)


def test_fused_traversal_edge_cases(vr):
    """Camera inside the volume, a volume behind the camera, tiny frames, axis-aligned orthographic
    rays, a step longer than the volume, and one brick (fused == sort-last bit for bit)."""
    cube = synth.Cube(29, 40, 36, 30, 3)
    data = cube.fill_host()
    g, _ = make_pair(cube, 16, 1, data=data)
    one = oracle.Volume(40, 36, 30, 64, 1, data=data)
    one.set_transfer_function(synth.tf_ramp(), synth.TF_VMIN, synth.TF_VMAX)
    g.set_traversal(vr.FUSED)
    W, H = 64, 48
    fr = synth.Framing(40, 36, 30, W, H)

    def both(view, proj, w, h, step, what):
        ref = one.render(view, proj, w, h, step, oracle.ALPHA)
        check_alpha(gpu_frame(g, view, proj, w, h, step, vr.ALPHA), ref, 0.99, what)
        check_mip(gpu_frame(g, view, proj, w, h, step, vr.MIP), one.render(view, proj, w, h, step, oracle.MIP), what)

    both(synth.look_at((20.3, 18.1, 14.2), (60, 40, 22), (0, 0, 1)), synth.perspective(70, W / H, 0.25, 200.0), W, H, 0.5, "inside")
    behind = synth.look_at((20, 18, 300), (20, 18, 600), (0, 1, 0))
    for mode in (vr.ALPHA, vr.MIP):
        assert not gpu_frame(g, behind, synth.perspective(40, W / H, 1.0, 100.0), W, H, 0.5, mode).any()
    for (w, h) in ((1, 1), (3, 2), (33, 5)):
        f2 = synth.Framing(40, 36, 30, w, h)
        both(f2.seeded(1, 0), f2.proj(False), w, h, 0.5, "%dx%d" % (w, h))
    both(synth.look_at((20, 18, -10.0), (20, 18, 0.0), (0.0, 1.0, 0.0)), synth.orthographic(20, 18, 1.0, 60.0), 40, 36, 1.0, "axis-aligned")
    for step in (200.0, 0.1):
        both(fr.seeded(1, 1), fr.proj(True), W, H, step, "step %g" % step)
    g1, _ = make_pair(cube, 64, 1, data=data)
    a = gpu_frame(g1, fr.turntable(3), fr.proj(False), W, H, 0.5, vr.ALPHA)
    g1.set_traversal(vr.FUSED)
    assert np.array_equal(gpu_frame(g1, fr.turntable(3), fr.proj(False), W, H, 0.5, vr.ALPHA), a)


# --------------------------------------------------------------------------- blanked voxels (R14)
def test_nan_voxels_are_blanked(vr):
    """NaN voxels (blanked channels, masked edges: the usual state of a radio cube) drop exactly the
    samples that rest on them on both sides: parity in both modes and traversals, with the same
    sample count (up to the samples that sit on the NaN-weight limit); the data range ignores them; culling and macro-cell skipping stay exact."""
    nx, ny, nz, B = 90, 70, 52, 16
    data = synth.Cube(91, nx, ny, nz, 8).fill_host()
    data[:, :, :5] = np.nan                       # a masked edge
    data[20:23] = np.nan                          # three blanked channels (across every brick column)
    data[30:47, 10:35, 40:70] = np.nan            # a masked box straddling brick seams
    rng = np.random.default_rng(5)
    data[rng.random(data.shape) < 0.002] = np.nan  # isolated bad voxels
    g = vr.Volume(nx, ny, nz, B, 1)
    g.upload(data)
    o = oracle.Volume(nx, ny, nz, B, 1, data=data)
    one = oracle.Volume(nx, ny, nz, 128, 1, data=data)
    assert g.minmax() == o.brick_minmax(-1) == (np.nanmin(data), np.nanmax(data))
    mm = g.debug_brick_minmax()
    for b in range(0, g.nbricks, 7):
        assert tuple(mm[b]) == o.brick_minmax(b)
    W, H = 180, 140
    fr = synth.Framing(nx, ny, nz, W, H)
    view, proj = fr.seeded(12, 0), fr.proj(False)
    g.set_counting(1)
    for tf_name, tf in (("translucent", synth.tf_translucent()), ("threshold", synth.tf_threshold())):
        for v in (g, o, one):
            v.set_transfer_function(tf, synth.TF_VMIN, synth.TF_VMAX)
            v.set_early_termination(2.0)          # no early termination: sample counts are exact
        for trav, orc in ((vr.SORT_LAST, o), (vr.FUSED, one)):
            g.set_traversal(trav)
            g.set_culling(False)
            ref = orc.render(view, proj, W, H, 0.5, oracle.ALPHA)
            img = gpu_frame(g, view, proj, W, H, 0.5, vr.ALPHA)
            assert np.isfinite(img).all()
            check_alpha(img, ref, 2.0, "NaN " + tf_name)
            slack = 4 * int(((ref["flags"] & oracle.FLAG_NAN_MARGIN) != 0).sum())   # samples on the NaN-weight limit may go either way
            assert abs(g.debug_stats()["samples"] - int(ref["counts"][..., 0].sum())) <= slack
            g.set_culling(True)
            assert np.array_equal(gpu_frame(g, view, proj, W, H, 0.5, vr.ALPHA), img)
            refm = orc.render(view, proj, W, H, 0.5, oracle.MIP)
            imgm = gpu_frame(g, view, proj, W, H, 0.5, vr.MIP)
            check_mip(imgm, refm, "NaN MIP")
            assert abs(g.debug_stats()["samples"] - int(refm["counts"][..., 0].sum())) <= slack
    # a fully blanked volume renders nothing
    gb = vr.Volume(24, 24, 24, 16, 1)
    gb.upload(np.full((24, 24, 24), np.nan, dtype=np.float32))
    gb.set_transfer_function(synth.tf_ramp(), synth.TF_VMIN, synth.TF_VMAX)
    f2 = synth.Framing(24, 24, 24, 48, 48)
    for mode in (vr.ALPHA, vr.MIP):
        assert not gpu_frame(gb, f2.seeded(1, 0), f2.proj(False), 48, 48, 0.5, mode).any()


# --------------------------------------------------------------------------- randomised configurations
@pytest.mark.parametrize("case", range(int(__import__("os").environ.get("VR_RANDOM_CASES", "64"))))
def test_randomised_configurations(vr, case):
    """Seeded random volumes, bricks, ghosts, steps (incl. the per-ray step), cameras (incl. eyes
    inside the volume), transfer functions, data kinds and blanked voxels, both modes and both
    traversals, culling on: parity with the oracle every time."""
    rng = np.random.default_rng(1000 + case)
    nx, ny, nz = (int(v) for v in rng.integers(18, 75, 3))
    brick = int(rng.choice([8, 12, 16, 20, 32, 64]))
    ghost = int(rng.choice([1, 1, 2])) if case % 7 else 0   # every seventh case without ghost cells (clamped fetches, seams as the oracle's)
    kind = int(rng.choice([0, 0, 1]))
    cube = synth.Cube(500 + case, nx, ny, nz, int(rng.integers(1, 8)), kind=kind)
    data = cube.fill_host()
    if rng.random() < 0.4:
        data[rng.random(data.shape) < 0.01] = np.nan
        a, b = sorted(int(v) for v in rng.integers(0, nz, 2))
        data[a:b + 1, : ny // 3] = np.nan
    if kind == 1:
        tf, lo, hi = synth.tf_density(), 0.0, synth.NBODY_VMAX
    else:
        tf = [synth.tf_ramp, synth.tf_translucent, synth.tf_threshold][int(rng.integers(0, 3))]()
        lo, hi = synth.TF_VMIN, synth.TF_VMAX
    tau = float(rng.choice([0.99, 0.9, 2.0]))
    step = float(rng.choice([0.0, 0.37, 0.5, 1.0, 1.63]))
    W, H = int(rng.integers(40, 130)), int(rng.integers(30, 100))
    fr = synth.Framing(nx, ny, nz, W, H)
    if rng.random() < 0.25:   # an eye inside the volume, looking at a random corner
        eye = (nx * rng.uniform(0.2, 0.8), ny * rng.uniform(0.2, 0.8), nz * rng.uniform(0.2, 0.8))
        corner = (nx * float(rng.integers(0, 2)), ny * float(rng.integers(0, 2)), nz * float(rng.integers(0, 2)))
        view, proj = synth.look_at(eye, corner, (0.0, 0.3, 1.0)), synth.perspective(60, W / H, 0.3, 400.0)
    else:
        view, proj = fr.seeded(700 + case, case), fr.proj(bool(rng.integers(0, 2)))
    linear = case % 5 == 3   # every fifth case on the x-linear comparison layout (hand-rolled sampler only)
    g = vr.Volume(nx, ny, nz, brick, ghost, layout=vr.LAYOUT_LINEAR) if linear else vr.Volume(nx, ny, nz, brick, ghost)
    g.upload(data)
    o = oracle.Volume(nx, ny, nz, brick, ghost, data=data)
    one = oracle.Volume(nx, ny, nz, 128, 1, data=data)
    for v in (g, o, one):
        v.set_transfer_function(tf, lo, hi)
        v.set_early_termination(tau)
    assert np.array_equal(g.debug_brick_order(view, proj), o.brick_order(view, proj))
    # the fused traversal has the one-brick oracle as its reference, which needs ghost cells (R17: no seams)
    for trav, orc in ((vr.SORT_LAST, o), (vr.FUSED, one)) if ghost > 0 else ((vr.SORT_LAST, o),):
        g.set_traversal(trav)
        ref = orc.render(view, proj, W, H, step, oracle.ALPHA)
        check_alpha(gpu_frame(g, view, proj, W, H, step if step > 0 else vr.STEP_AUTO, vr.ALPHA), ref,
                    tau, "case %d" % case)
        refm = orc.render(view, proj, W, H, step, oracle.MIP)
        got = gpu_frame(g, view, proj, W, H, step if step > 0 else vr.STEP_AUTO, vr.MIP)
        check_mip(got, refm, "case %d" % case)
    if linear:
        with pytest.raises(vr.VrError):
            g.set_sampler(vr.SAMPLER_TEXTURE)
        return
    # R23: MIP through the texture arrays of any texel width is the hand-rolled frame, bit for bit
    g.set_traversal(vr.SORT_LAST)
    want = gpu_frame(g, view, proj, W, H, step if step > 0 else vr.STEP_AUTO, vr.MIP)
    for s in (vr.SAMPLER_TEXTURE, vr.SAMPLER_TEXTURE_HALF, vr.SAMPLER_TEXTURE_BYTE):
        g.set_sampler(s)
        assert np.array_equal(gpu_frame(g, view, proj, W, H, step if step > 0 else vr.STEP_AUTO, vr.MIP), want), (case, s)
    # R20 / R22: ALPHA values through float32 and float16 texels against the same oracle at the same 2e-3 (R12's band widened
    # to the filter's error); stepped tables and blanked bricks fall back to the hand-rolled sampler inside the library
    # the band: the filter moves a ray's transmittance by up to ~4e-3 of itself, i.e. A_b near tau by 4e-3 (1 - tau); 5x that
    o.set_ert_margin(0.02 * (1.0 - tau) if tau < 1.0 else 2e-4)
    ref = o.render(view, proj, W, H, step, oracle.ALPHA)
    for s in (vr.SAMPLER_TEXTURE, vr.SAMPLER_TEXTURE_HALF):
        g.set_sampler(s)
        check_alpha(gpu_frame(g, view, proj, W, H, step if step > 0 else vr.STEP_AUTO, vr.ALPHA), ref, tau,
                    "case %d sampler %d" % (case, s), envelope=True, max_flagged=1.0)
    # ... and the fused traversal through the float32 arrays (per-lane texture objects) against the one-brick oracle
    if ghost == 0:
        return
    one.set_ert_margin(0.02 * (1.0 - tau) if tau < 1.0 else 2e-4)
    g.set_sampler(vr.SAMPLER_TEXTURE)
    g.set_traversal(vr.FUSED)
    check_alpha(gpu_frame(g, view, proj, W, H, step if step > 0 else vr.STEP_AUTO, vr.ALPHA), one.render(view, proj, W, H, step, oracle.ALPHA),
                tau, "case %d fused through the arrays" % case, envelope=True, max_flagged=1.0)


# --------------------------------------------------------------------------- state across calls
def test_handle_state_survives_a_session(vr):
    """Two handles alive at once; frame sizes that grow and shrink (scratch regrown), a sub-box
    re-upload in the middle (range tables invalidated), transfer-function, traversal and culling
    switches, device, host and pipelined host frames interleaved: every frame equals the frame a
    FRESH handle renders from the same state, bit for bit."""
    import torch
    ca, cb = synth.Cube(81, 72, 60, 48, 5), synth.Cube(82, 40, 56, 64, 3, kind=synth.NBODY)
    da, db = ca.fill_host(), cb.fill_host()
    ga, gb = vr.Volume(72, 60, 48, 16, 1), vr.Volume(40, 56, 64, 32, 1)
    ga.upload(da)
    gb.upload(db)
    tfs = {"ramp": (synth.tf_ramp(), synth.TF_VMIN, synth.TF_VMAX), "thr": (synth.tf_threshold(), synth.TF_VMIN, synth.TF_VMAX),
           "dens": (synth.tf_density(), 0.0, synth.NBODY_VMAX)}
    ga.set_transfer_function(*tfs["ramp"])
    gb.set_transfer_function(*tfs["dens"])
    state = {"a": dict(data=da, dims=(72, 60, 48), brick=16, tf="ramp", trav=vr.SORT_LAST, cull=True),
             "b": dict(data=db, dims=(40, 56, 64), brick=32, tf="dens", trav=vr.SORT_LAST, cull=True)}
    handles = {"a": ga, "b": gb}

    def fresh(which, W, H, k, mode):
        st = state[which]
        g = vr.Volume(*st["dims"], st["brick"], 1)
        g.upload(st["data"])
        g.set_transfer_function(*tfs[st["tf"]])
        g.set_traversal(st["trav"])
        g.set_culling(st["cull"])
        fr = synth.Framing(*st["dims"], W, H)
        return gpu_frame(g, fr.seeded(3, k), fr.proj(k % 2 == 1), W, H, 0.5, mode)

    def frame(which, W, H, k, mode, how):
        g, st = handles[which], state[which]
        fr = synth.Framing(*st["dims"], W, H)
        view, proj = fr.seeded(3, k), fr.proj(k % 2 == 1)
        if how == "device":
            return gpu_frame(g, view, proj, W, H, 0.5, mode)
        if how == "host":
            return g.render_host(view, proj, W, H, 0.5, mode).astype(np.float64)
        buf = torch.empty((H, W, 4), dtype=torch.float32).pin_memory()
        g.render_host_async(view, proj, W, H, 0.5, mode, buf)
        g.render_host_wait()
        return buf.numpy().astype(np.float64)

    script = [("a", 96, 64, 0, vr.ALPHA, "device"), ("b", 160, 120, 1, vr.MIP, "async"), ("a", 200, 150, 2, vr.MIP, "host"),
              ("tf", "a", "thr"), ("a", 64, 48, 3, vr.ALPHA, "async"), ("b", 80, 60, 4, vr.ALPHA, "device"),
              ("trav", "a", vr.FUSED), ("a", 120, 90, 5, vr.ALPHA, "device"), ("upload", "a"), ("a", 120, 90, 6, vr.ALPHA, "host"),
              ("cull", "b", False), ("b", 160, 120, 7, vr.MIP, "device"), ("trav", "a", vr.SORT_LAST), ("tf", "a", "ramp"),
              ("a", 210, 130, 8, vr.ALPHA, "device"), ("cull", "b", True), ("trav", "b", vr.FUSED), ("b", 33, 17, 9, vr.ALPHA, "async"),
              ("a", 96, 64, 10, vr.MIP, "device")]
    for op in script:
        if op[0] == "tf":
            handles[op[1]].set_transfer_function(*tfs[op[2]])
            state[op[1]]["tf"] = op[2]
        elif op[0] == "trav":
            handles[op[1]].set_traversal(op[2])
            state[op[1]]["trav"] = op[2]
        elif op[0] == "cull":
            handles[op[1]].set_culling(op[2])
            state[op[1]]["cull"] = op[2]
        elif op[0] == "upload":   # overwrite a box that straddles brick seams with bright values
            box = np.full((20, 22, 24), 7.0, dtype=np.float32)
            handles[op[1]].upload(box, origin=(10, 12, 14))
            d = state[op[1]]["data"].copy()
            d[14:34, 12:34, 10:34] = box
            state[op[1]]["data"] = d
        else:
            which, W, H, k, mode, how = op
            assert np.array_equal(frame(which, W, H, k, mode, how), fresh(which, W, H, k, mode)), op


# --------------------------------------------------------------------------- edge cases
def test_edge_cases(vr):
    import torch
    cube = synth.Cube(13, 20, 18, 16, 2)
    g, o = make_pair(cube, 8, 1)
    fr = synth.Framing(20, 18, 16, 64, 48)
    # 1x1 frame and a 3x2 frame
    for (W, H) in ((1, 1), (3, 2), (33, 5)):
        f2 = synth.Framing(20, 18, 16, W, H)
        view, proj = f2.seeded(1, 0), f2.proj(False)
        ref = o.render(view, proj, W, H, 0.5, oracle.ALPHA)
        check_alpha(gpu_frame(g, view, proj, W, H, 0.5, vr.ALPHA), ref, 0.99, "%dx%d" % (W, H))
    W, H = 64, 48
    # the volume is behind the camera / off screen: transparent black, both modes
    view = synth.look_at((10, 9, 200), (10, 9, 400), (0, 1, 0))
    proj = synth.perspective(40, W / H, 1.0, 100.0)
    for mode in (vr.ALPHA, vr.MIP):
        assert not gpu_frame(g, view, proj, W, H, 0.5, mode).any()
    # camera inside the volume (R2: the ray starts on the near plane)
    view = synth.look_at((10.3, 9.1, 8.2), (30, 20, 12), (0, 0, 1))
    proj = synth.perspective(70, W / H, 0.25, 100.0)
    ref = o.render(view, proj, W, H, 0.5, oracle.ALPHA)
    check_alpha(gpu_frame(g, view, proj, W, H, 0.5, vr.ALPHA), ref, 0.99, "inside")
    ref = o.render(view, proj, W, H, 0.5, oracle.MIP)
    check_mip(gpu_frame(g, view, proj, W, H, 0.5, vr.MIP), ref, "inside")
    # a step longer than the volume: one (clipped) sample per ray; and a fine step
    view, proj = fr.seeded(1, 1), fr.proj(True)
    for step in (100.0, 0.1, 1.0):
        ref = o.render(view, proj, W, H, step, oracle.ALPHA)
        check_alpha(gpu_frame(g, view, proj, W, H, step, vr.ALPHA), ref, 0.99, "step %g" % step)
        ref = o.render(view, proj, W, H, step, oracle.MIP)
        check_mip(gpu_frame(g, view, proj, W, H, step, vr.MIP), ref, "step %g" % step)
    # axis-aligned orthographic view: two direction components are exactly zero (R4)
    view = synth.look_at((10, 9, -10.0), (10, 9, 0.0), (0.0, 1.0, 0.0))
    proj = synth.orthographic(10, 9, 1.0, 46.0)
    ref = o.render(view, proj, 20, 18, 1.0, oracle.MIP)
    check_mip(gpu_frame(g, view, proj, 20, 18, 1.0, vr.MIP), ref, "axis-aligned")
    ref = o.render(view, proj, 20, 18, 1.0, oracle.ALPHA)
    check_alpha(gpu_frame(g, view, proj, 20, 18, 1.0, vr.ALPHA), ref, 0.99, "axis-aligned")
    # host-memory entry gives the same frame
    view, proj = fr.seeded(1, 2), fr.proj(False)
    a = gpu_frame(g, view, proj, W, H, 0.5, vr.ALPHA)
    b = g.render_host(view, proj, W, H, 0.5, vr.ALPHA)
    assert np.array_equal(a.astype(np.float32), b)
    pinned = torch.empty((H, W, 4), dtype=torch.float32).pin_memory()
    g.render_host(view, proj, W, H, 0.5, vr.ALPHA, out=pinned)
    assert np.array_equal(pinned.numpy(), b)


def test_errors(vr):
    import torch
    g = vr.Volume(16, 16, 16, 8, 1)
    out = torch.empty((8, 8, 4), dtype=torch.float32, device="cuda")
    I = np.eye(4, dtype=np.float32).T.reshape(16)
    with pytest.raises(vr.VrError) as e:
        g.render(I, I, 8, 8, 0.5, vr.ALPHA, out)
    assert e.value.status == 4  # no transfer function
    g.set_transfer_function(synth.tf_ramp(), -3, 10)
    with pytest.raises(vr.VrError) as e:
        g.render(I, I, 8, 8, 0.5, vr.ALPHA, out)
    assert e.value.status == 4  # nothing uploaded
    g.upload(np.zeros((16, 16, 16), dtype=np.float32))
    with pytest.raises(vr.VrError) as e:
        g.render(I, I, 8, 8, -0.5, vr.ALPHA, out)   # 0 is VR_STEP_AUTO; negative and NaN steps are errors
    assert e.value.status == 1
    with pytest.raises(vr.VrError) as e:
        g.render(I, I, 8, 8, float("nan"), vr.ALPHA, out)
    assert e.value.status == 1
    with pytest.raises(vr.VrError) as e:
        g.render(I, np.zeros(16, dtype=np.float32), 8, 8, 0.5, vr.ALPHA, out)
    assert e.value.status == 1 and "singular" in str(e.value)
    with pytest.raises(vr.VrError):
        g.render(I, I, 8, 8, 0.5, 7, out)
    with pytest.raises(vr.VrError):
        g.set_transfer_function(synth.tf_ramp(), 1.0, 1.0)
    with pytest.raises(vr.VrError):
        g.upload(np.zeros((4, 4, 4), dtype=np.float32), origin=(14, 0, 0))
    bad = synth.tf_ramp()
    bad[7, 3] = 1.5   # an opacity outside [0,1] would turn log2(1 - a) into NaN: refused, on both sides
    with pytest.raises(vr.VrError) as e:
        g.set_transfer_function(bad, -3, 10)
    assert e.value.status == 1 and "alpha" in str(e.value)
    with pytest.raises(ValueError):
        oracle.Volume(16, 16, 16, 8, 1).set_transfer_function(bad, -3, 10)
    with pytest.raises(ValueError):   # the binding's own argument checks raise (they are not asserts)
        g.render(I, I, 8, 8, 0.5, vr.ALPHA, torch.empty((4, 4, 4), dtype=torch.float32, device="cuda"))
    g.render(I, I, 8, 8, 0.5, vr.ALPHA, out)  # still usable after errors
    torch.cuda.synchronize()


def test_environment_knobs_are_validated(vr, monkeypatch):
    monkeypatch.setenv("VR_TILE", "9,9,9")
    with pytest.raises(vr.VrError) as e:
        vr.Volume(16, 16, 16, 8, 1)
    assert e.value.status == 1 and "VR_TILE" in str(e.value)
    monkeypatch.setenv("VR_TILE", "3,3,3,0,0,0")   # 512 cells: not one 128-byte line
    with pytest.raises(vr.VrError):
        vr.Volume(16, 16, 16, 8, 1)
    monkeypatch.delenv("VR_TILE")
    monkeypatch.setenv("VR_LAYOUT", "tiled")
    with pytest.raises(vr.VrError) as e:
        vr.Volume(16, 16, 16, 8, 1)
    assert "VR_LAYOUT" in str(e.value)


def test_reserved_views_render_without_allocating_and_torch_allocator(vr):
    """vr_reserve_views sizes every per-view buffer up front (vr_render then never allocates: the device's free memory
    does not move); a view that was not announced and needs more scratch still renders. With vr_set_allocator the
    library's buffers come out of torch's caching allocator (north_star: PyTorch for device memory)."""
    import torch
    cube = synth.Cube(41, 96, 80, 64, 6)
    data = cube.fill_host()
    W, H = 320, 200
    fr = synth.Framing(cube.nx, cube.ny, cube.nz, W, H)
    views = [fr.turntable(k) for k in range(0, 36, 3)]
    projs = [fr.proj(False)] * len(views)
    import gc
    gc.collect()
    torch.cuda.synchronize()
    before = torch.cuda.memory_allocated()
    vr.use_torch_allocator(True)
    try:
        g = vr.Volume(cube.nx, cube.ny, cube.nz, 32, 1)
    finally:
        vr.use_torch_allocator(False)
    held = torch.cuda.memory_allocated() - before
    assert held >= 18 * 9 * 9 * 17 * 128  # at least the brick store (18 slots of 9 x 9 x 17 micro-tiles of 128 bytes) is torch's
    o = oracle.Volume(cube.nx, cube.ny, cube.nz, 32, 1, data=data)
    g.upload(torch.from_numpy(data).cuda())
    for v in (g, o):
        v.set_transfer_function(synth.tf_ramp(), synth.TF_VMIN, synth.TF_VMAX)
    g.reserve_views(views, projs, W, H)
    host = torch.empty((H, W, 4), dtype=torch.float32).pin_memory()
    out = torch.empty((H, W, 4), dtype=torch.float32, device="cuda")
    torch.cuda.synchronize()
    # the handle allocates through torch: any block it took would be counted here (a cumulative count of allocations:
    # tensors of earlier tests being collected meanwhile cannot disturb it)
    allocs0 = torch.cuda.memory_stats()["allocation.all.allocated"]
    for view in views:
        g.render(view, projs[0], W, H, 0.5, vr.ALPHA, out)
        g.render(view, projs[0], W, H, 0.5, vr.MIP, out)
        g.render_host_async(view, projs[0], W, H, 0.5, vr.ALPHA, host)
    g.render_host_wait()
    g.render_host(views[0], projs[0], W, H, 0.5, vr.ALPHA, host.numpy())
    torch.cuda.synchronize()
    assert torch.cuda.memory_stats()["allocation.all.allocated"] == allocs0
    ref = o.render(views[0], projs[0], W, H, 0.5, oracle.ALPHA)
    check_alpha(host.numpy().astype(np.float64), ref, 0.99, "reserved views")
    # an unannounced, much closer view needs more sub-image scratch: it grows (and renders correctly)
    close = synth.look_at((cube.nx * 0.5, cube.ny * 0.5, cube.nz * 1.2), (cube.nx * 0.5, cube.ny * 0.5, 0.0), (0, 1, 0))
    wide = synth.perspective(100.0, W / H, 0.5, 500.0)
    img = gpu_frame(g, close, wide, W, H, 0.5, vr.ALPHA)
    check_alpha(img, o.render(close, wide, W, H, 0.5, oracle.ALPHA), 0.99, "unannounced view")
    g.close()
    torch.cuda.synchronize()
    assert torch.cuda.memory_allocated() - before < held  # the handle's buffers went back to torch


# --------------------------------------------------------------------------- a9 stand-alone
@pytest.mark.parametrize("case", range(int(__import__("os").environ.get("VR_COMPOSITE_CASES", "16"))))
def test_randomised_compositing(vr, case):
    """Row a9 under random use: 0-40 layers with random rectangles (empty, one pixel, full frame, straddling tile borders),
    random visibility orders, frames that are not multiples of the 32x8 tile: vr_composite and vr_composite_static against
    the oracle (R15, 1e-5) and against each other (bit-identical)."""
    import torch
    rng = np.random.default_rng(11000 + case)
    W, H = int(rng.integers(1, 300)), int(rng.integers(1, 200))
    n = int(rng.integers(0, 41))
    rects, layers_h = [], []
    for l in range(n):
        kind = rng.random()
        if kind < 0.1:
            x0, y0, x1, y1 = 0, 0, W, H
        elif kind < 0.2:
            x0 = x1 = int(rng.integers(0, W + 1)); y0, y1 = 0, H          # empty
        else:
            x0, y0 = int(rng.integers(0, W)), int(rng.integers(0, H))
            x1, y1 = int(rng.integers(x0, W + 1)), int(rng.integers(y0, H + 1))
        rects.append((x0, y0, x1, y1))
        a = rng.random((y1 - y0, x1 - x0, 1)).astype(np.float32)
        layers_h.append(np.concatenate([rng.random((y1 - y0, x1 - x0, 3)).astype(np.float32) * a, a], axis=-1))
    order = rng.permutation(n).astype(np.int32)
    ref = oracle.composite(layers_h, rects, order, W, H)
    layers_d = [torch.from_numpy(l).cuda() if l.size else torch.empty((0, 0, 4), device="cuda") for l in layers_h]
    out = torch.full((H, W, 4), 7.0, dtype=torch.float32, device="cuda")
    out_s = torch.full((H, W, 4), -7.0, dtype=torch.float32, device="cuda")
    vr.composite(layers_d, np.array(rects, dtype=np.int32).reshape(n, 4), order, W, H, out)
    vr.composite_static(layers_d, np.array(rects, dtype=np.int32).reshape(n, 4), order, W, H, out_s)
    torch.cuda.synchronize()
    assert np.abs(out.cpu().numpy() - ref).max() < 1e-5, case
    assert torch.equal(out, out_s), case


def test_composite_matches_oracle(vr):
    import torch
    W, H, n = 97, 61, 9
    rects, layers_h = [], []
    for l in range(n):
        x0, y0 = int(synth.u01(1, 1, l) * 60), int(synth.u01(1, 2, l) * 40)
        x1, y1 = min(W, x0 + 5 + int(synth.u01(1, 3, l) * 70)), min(H, y0 + 3 + int(synth.u01(1, 4, l) * 50))
        if l == 0:
            x0, y0, x1, y1 = 0, 0, W, H
        if l == 1:
            x1 = x0  # an empty layer
        rects.append((x0, y0, x1, y1))
        layers_h.append(synth.layer_host(99, l, 0, (x1 - x0) * (y1 - y0)).reshape(y1 - y0, x1 - x0, 4))
    order = synth.permutation(5, n)
    ref = oracle.composite(layers_h, rects, order, W, H)
    out = torch.full((H, W, 4), 7.0, dtype=torch.float32, device="cuda")
    layers_d = [torch.from_numpy(l).cuda() if l.size else torch.empty((0, 0, 4), device="cuda") for l in layers_h]
    vr.composite(layers_d, rects, order, W, H, out)
    torch.cuda.synchronize()
    assert np.abs(out.cpu().numpy() - ref).max() < 1e-5  # R15
    with pytest.raises(vr.VrError):
        vr.composite(layers_d, rects, np.zeros(n, dtype=np.int32), W, H, out)  # not a permutation
