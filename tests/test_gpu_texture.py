"""GPU parity of the texture-object arm of rows a1 / a5 (vr_set_sampler(VR_SAMPLER_TEXTURE)
"built-in tri-linear interpolation"): VR_ALPHA frames through hardware-filtered 3-D CUDA arrays against the same
oracle at north_star's 2e-3. The sample SET is the hand-rolled path's (same FP64 set-up); the filter's 8-bit
weights move a brick's accumulated opacity by up to ~1e-4, so a termination test within 2e-4 of tau may go either
way: such pixels are flagged by the oracle (R12, margin widened to 2e-4) and must lie within 2e-3 of the interval
between the oracle's frames for tau - 2e-4 and tau + 2e-4."""
import numpy as np
import pytest

import oracle
import synth
from helpers import check_alpha, check_mip, gpu_frame, make_pair, seeded_pixels

pytestmark = pytest.mark.gpu
TEX_MARGIN = 2e-4


@pytest.fixture(scope="module")
def vr(cuda_device):
    from paper_1205_0282_b200 import build
    build.build()
    import paper_1205_0282_b200 as vr
    return vr


TEXELS = ["float32", "float16"]  # the arrays ALPHA frames may take their values from


def tex_pair(vr, cube, brick, ghost=1, tf=None, tau=0.99, data=None, texels="float32"):
    g, o = make_pair(cube, brick, ghost, tf=tf, tau=tau, data=data)
    g.set_sampler(vr.SAMPLER_TEXTURE if texels == "float32" else vr.SAMPLER_TEXTURE_HALF)
    o.set_ert_margin(TEX_MARGIN)
    return g, o


@pytest.mark.parametrize("texels", TEXELS)
@pytest.mark.parametrize("tf_name", ["ramp", "translucent"])
def test_config0_full_frames_texture(vr, tf_name, texels):
    c = synth.CONFIGS["c0"]
    cube = synth.config_cube("c0")
    tf = synth.tf_ramp() if tf_name == "ramp" else synth.tf_translucent()
    g, o = tex_pair(vr, cube, c["brick"], c["ghost"], tf=tf, texels=texels)
    W, H = c["width"], c["height"]
    fr = synth.Framing(cube.nx, cube.ny, cube.nz, W, H)
    worst = 0.0
    for ortho in (False, True):
        for k in range(3):
            view, proj = fr.seeded(77, k), fr.proj(ortho)
            ref = o.render(view, proj, W, H, c["step"], oracle.ALPHA)
            img = gpu_frame(g, view, proj, W, H, c["step"], vr.ALPHA)
            worst = max(worst, check_alpha(img, ref, 0.99, "c0 texture %s %d" % (tf_name, k), envelope=True, max_flagged=1.0))
            # unflagged pixels alone: the plain 2e-3 bound, and the filter's weights do show (not the manual path)
            un = (ref["flags"] & oracle.FLAG_ERT_MARGIN) == 0
            assert np.abs(img - ref["image"]).max(axis=-1)[un].max() <= 2e-3
    g.set_sampler(vr.SAMPLER_MANUAL)
    man = gpu_frame(g, view, proj, W, H, c["step"], vr.ALPHA)
    assert 1e-7 < np.abs(man - img).max() < 0.02  # two different samplers, the same picture


@pytest.mark.parametrize("texels", TEXELS)
@pytest.mark.parametrize("ghost,tau", [(1, 0.99), (1, 2.0), (2, 0.99), (0, 2.0)])
def test_bricked_ragged_texture_frames_subimages_and_counts(vr, ghost, tau, texels):
    """Ragged multi-brick volume: frames, each brick's sub-image, and - with early termination off - exactly the
    hand-rolled path's sample count; ghost = 0 relies on the arrays' clamp addressing (seams as the oracle's)."""
    cube = synth.Cube(11, 100, 90, 70, 12)
    tf = synth.tf_translucent() if tau > 1 else synth.tf_ramp()
    g, o = tex_pair(vr, cube, 32, ghost, tf=tf, tau=tau, texels=texels)
    W, H = 203, 117
    fr = synth.Framing(cube.nx, cube.ny, cube.nz, W, H)
    pix = seeded_pixels(4, W, H, 300)
    g.set_counting(1)
    for k, ortho in ((0, False), (1, True)):
        view, proj = fr.seeded(77, k), fr.proj(ortho)
        ref = o.render(view, proj, W, H, 0.5, oracle.ALPHA)
        img = gpu_frame(g, view, proj, W, H, 0.5, vr.ALPHA)
        n_tex = g.debug_stats()["samples"]
        check_alpha(img, ref, tau, "texture ghost %d view %d" % (ghost, k), envelope=True, max_flagged=1.0)
        sub_ref = o.render(view, proj, W, H, 0.5, oracle.ALPHA, pixels=pix, want_sub=True)
        check_alpha(g.debug_subimages(pix).astype(np.float64), sub_ref, tau, "texture sub-images", key="sub", envelope=True,
                    max_flagged=1.0)
        if tau > 1:
            assert n_tex == int(ref["counts"][..., 0].sum())
        # MIP frames are exact through the arrays too (candidates re-evaluated by hand): bit-identical with the sampler switched back
        m_tex = gpu_frame(g, view, proj, W, H, 0.5, vr.MIP)
        g.set_sampler(vr.SAMPLER_MANUAL)
        assert np.array_equal(gpu_frame(g, view, proj, W, H, 0.5, vr.MIP), m_tex)
        g.set_sampler(vr.SAMPLER_TEXTURE if texels == "float32" else vr.SAMPLER_TEXTURE_HALF)
        check_mip(m_tex, o.render(view, proj, W, H, 0.5, oracle.MIP), "MIP beside the texture arm")


def test_texture_arm_follows_uploads_and_blanked_voxels(vr):
    """The arrays are refilled after an upload; NaN voxels (R14) go through the exact rule of the float32 store."""
    import torch
    cube = synth.Cube(31, 72, 40, 56, 6)
    data = cube.fill_host()
    g, o = tex_pair(vr, cube, 32, 1, tf=synth.tf_translucent(), tau=2.0, data=data)
    W, H = 144, 100
    fr = synth.Framing(cube.nx, cube.ny, cube.nz, W, H)
    view, proj = fr.turntable(5), fr.proj(False)
    check_alpha(gpu_frame(g, view, proj, W, H, 0.5, vr.ALPHA), o.render(view, proj, W, H, 0.5, oracle.ALPHA), 2.0, "first upload")
    d2 = data.copy()
    d2[10:30, 5:25, 20:50] = np.nan      # a blanked box across brick seams
    d2[40:, :, :8] = np.nan              # a blanked edge
    d2[3, 7, 60] = np.nan                # an isolated bad voxel
    d2[31:34, 20:22, 30:33] += 4.0
    g.upload(torch.from_numpy(d2).cuda())
    o2 = oracle.Volume(cube.nx, cube.ny, cube.nz, 32, 1, data=d2)
    o2.set_transfer_function(synth.tf_translucent(), synth.TF_VMIN, synth.TF_VMAX)
    o2.set_early_termination(2.0)
    g.set_counting(1)
    ref = o2.render(view, proj, W, H, 0.5, oracle.ALPHA)
    img = gpu_frame(g, view, proj, W, H, 0.5, vr.ALPHA)
    assert np.isfinite(img).all()
    check_alpha(img, ref, 2.0, "second upload, blanked voxels")
    slack = 4 * int(((ref["flags"] & oracle.FLAG_NAN_MARGIN) != 0).sum())
    assert abs(g.debug_stats()["samples"] - int(ref["counts"][..., 0].sum())) <= slack
    assert np.abs(img - o.render(view, proj, W, H, 0.5, oracle.ALPHA)["image"]).max() > 1e-2  # not the first cube's frame


def test_texture_arm_keeps_stepped_tables_on_the_hand_rolled_path_and_errors(vr):
    """A transfer function with a step (threshold, toe) is outside what 8-bit filter weights can render to 2e-3
    (measured 8e-2): such frames keep the hand-rolled sampler, bit for bit, also with macro-cell skipping; a smooth
    table with a transparent range (three zero entries, then a gentle ramp) does use the texture arm with skipping."""
    cube = synth.Cube(33, 96, 80, 64, 10)
    g, o = tex_pair(vr, cube, 32, 1, tf=synth.tf_threshold())
    W, H = 160, 120
    fr = synth.Framing(cube.nx, cube.ny, cube.nz, W, H)
    view, proj = fr.seeded(9, 0), fr.proj(False)
    tex_frame = gpu_frame(g, view, proj, W, H, 0.5, vr.ALPHA)
    g.set_sampler(vr.SAMPLER_MANUAL)
    assert np.array_equal(gpu_frame(g, view, proj, W, H, 0.5, vr.ALPHA), tex_frame)
    g.set_sampler(vr.SAMPLER_TEXTURE)
    check_alpha(tex_frame, o.render(view, proj, W, H, 0.5, oracle.ALPHA), 0.99, "threshold table")
    # smooth table with a transparent range: alpha = max(0, u - 0.55) (zero below 4.2 sigma, then the ramp's slope: no
    # step), colours = u
    tf = synth.tf_ramp()
    tf[:, 3] = np.maximum(0.0, tf[:, 3] - 0.55)
    for v in (g, o):
        v.set_transfer_function(tf, synth.TF_VMIN, synth.TF_VMAX)
    g.set_counting(1)
    on = gpu_frame(g, view, proj, W, H, 0.5, vr.ALPHA)
    n_on = g.debug_stats()["samples"]
    g.set_culling(False)
    off = gpu_frame(g, view, proj, W, H, 0.5, vr.ALPHA)
    n_off = g.debug_stats()["samples"]
    assert np.array_equal(on, off) and n_on < n_off
    check_alpha(on, o.render(view, proj, W, H, 0.5, oracle.ALPHA), 0.99, "texture + skipping", envelope=True, max_flagged=1.0)
    g.set_sampler(vr.SAMPLER_MANUAL)
    assert 1e-7 < np.abs(gpu_frame(g, view, proj, W, H, 0.5, vr.ALPHA) - off).max() < 0.02  # the texture arm was in use
    lin = vr.Volume(32, 32, 32, 16, 1, layout=vr.LAYOUT_LINEAR)
    with pytest.raises(vr.VrError) as e:
        lin.set_sampler(vr.SAMPLER_TEXTURE)
    assert e.value.status == 4
    with pytest.raises(vr.VrError):
        g.set_sampler(7)


@pytest.mark.parametrize("texels", TEXELS)
@pytest.mark.parametrize("tau", [0.99, 2.0])
def test_fused_traversal_through_the_texture_arm(vr, tau, texels):
    """Row f2 with the texture sampler: one ray through all bricks, per-lane texture objects (the rays of a warp may be
    in different bricks), against the oracle holding the cube in ONE brick (R17); early termination off: exactly the
    hand-rolled path's sample count. A brick with blanked voxels takes the hand-rolled loop inside the same kernel."""
    import torch
    cube = synth.Cube(51, 100, 90, 70, 12)
    data = cube.fill_host()
    tf = synth.tf_translucent() if tau > 1 else synth.tf_ramp()
    g, _ = tex_pair(vr, cube, 32, 1, tf=tf, tau=tau, data=data, texels=texels)
    one = oracle.Volume(cube.nx, cube.ny, cube.nz, 128, 1, data=data)
    one.set_transfer_function(tf, synth.TF_VMIN, synth.TF_VMAX)
    one.set_early_termination(tau)
    one.set_ert_margin(TEX_MARGIN)
    W, H = 203, 117
    fr = synth.Framing(cube.nx, cube.ny, cube.nz, W, H)
    g.set_traversal(vr.FUSED)
    g.set_counting(1)
    for k, ortho in ((0, False), (1, True)):
        view, proj = fr.seeded(77, k), fr.proj(ortho)
        ref = one.render(view, proj, W, H, 0.5, oracle.ALPHA)
        img = gpu_frame(g, view, proj, W, H, 0.5, vr.ALPHA)
        n_tex = g.debug_stats()["samples"]
        check_alpha(img, ref, tau, "fused texture view %d" % k, envelope=True, max_flagged=1.0)
        if tau > 1:
            assert n_tex == int(ref["counts"][..., 0].sum())
        g.set_sampler(vr.SAMPLER_MANUAL)
        man = gpu_frame(g, view, proj, W, H, 0.5, vr.ALPHA)
        g.set_sampler(vr.SAMPLER_TEXTURE if texels == "float32" else vr.SAMPLER_TEXTURE_HALF)
        assert 1e-7 < np.abs(man - img).max() < 0.02
    # blanked voxels in two bricks: those bricks are sampled by hand, the rest through the arrays, in one frame
    d2 = data.copy()
    d2[5:20, 40:60, 10:30] = np.nan
    g.upload(torch.from_numpy(d2).cuda())
    one2 = oracle.Volume(cube.nx, cube.ny, cube.nz, 128, 1, data=d2)
    one2.set_transfer_function(tf, synth.TF_VMIN, synth.TF_VMAX)
    one2.set_early_termination(tau)
    one2.set_ert_margin(TEX_MARGIN)
    ref = one2.render(view, proj, W, H, 0.5, oracle.ALPHA)
    img = gpu_frame(g, view, proj, W, H, 0.5, vr.ALPHA)
    assert np.isfinite(img).all()
    check_alpha(img, ref, tau, "fused texture, blanked box", envelope=True, max_flagged=1.0)


@pytest.mark.parametrize("texels", TEXELS)
def test_released_store_renders_through_the_arrays_alone(vr, texels):
    """VR_LAYOUT_TILED_RELEASABLE + vr_volume_release_store (the texture arm for cubes whose second copy does not fit):
    frames before the release (texture sampler, both stores present) and after it (float32 cells handed back) agree
    (only a ray's exit samples come from the float32 store while it exists), match the oracle, the device gets the memory back, bricks with blanked voxels keep their float32
    cells and the exact R14 rule, and everything that needs the float32 store refuses."""
    import torch
    dims, brick = (160, 128, 96), 32
    cube = synth.Cube(61, *dims, 10)
    data = cube.fill_host()
    data[70:90, 40:60, 100:120] = np.nan          # blanked voxels in a few bricks
    W, H = 203, 117
    fr = synth.Framing(*dims, W, H)
    g = vr.Volume(*dims, brick, 1, layout=vr.LAYOUT_TILED_RELEASABLE)
    g.upload(torch.from_numpy(data).cuda())
    o = oracle.Volume(*dims, brick, 1, data=data)
    one = oracle.Volume(*dims, 256, 1, data=data)
    for v in (g, o, one):
        v.set_transfer_function(synth.tf_ramp(), synth.TF_VMIN, synth.TF_VMAX)
        v.set_early_termination(0.99)
    o.set_ert_margin(TEX_MARGIN)
    one.set_ert_margin(TEX_MARGIN)
    mip_before = gpu_frame(g, fr.seeded(3, 0), fr.proj(False), W, H, 0.5, vr.MIP)
    check_mip(mip_before, o.render(fr.seeded(3, 0), fr.proj(False), W, H, 0.5, oracle.MIP), "releasable handle, MIP before the release")
    g.set_sampler(vr.SAMPLER_TEXTURE if texels == "float32" else vr.SAMPLER_TEXTURE_HALF)  # the released arrays take this width
    views = [(fr.seeded(3, k), fr.proj(k == 1)) for k in range(2)]
    before = [gpu_frame(g, v, p, W, H, 1.0, vr.ALPHA) for v, p in views]
    lo, hi = g.minmax()
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    freed = g.release_store()
    torch.cuda.synchronize()
    store_bytes = g.nbricks * 9 * 9 * 17 * 128
    assert freed > 0.6 * store_bytes                                   # all but the blanked bricks (and the shared granules)
    assert torch.cuda.mem_get_info()[0] > free0 - 0.5 * store_bytes    # a second copy was NOT needed at any time ...
    assert g.minmax() == (lo, hi)                                      # ... and the range tables survive
    for (v, p), b in zip(views, before):
        after = gpu_frame(g, v, p, W, H, 1.0, vr.ALPHA)
        # the same arrays before and after; only the (at most two) exit samples of a ray came from the float32 store before
        assert np.abs(after - b).max() < 1e-3 and (after != b).mean() < 0.5
        check_alpha(after, o.render(v, p, W, H, 1.0, oracle.ALPHA), 0.99, "released store", envelope=True, max_flagged=1.0)
    g.set_traversal(vr.FUSED)
    fused = gpu_frame(g, *views[0], W, H, 1.0, vr.ALPHA)
    check_alpha(fused, one.render(*views[0], W, H, 1.0, oracle.ALPHA), 0.99, "released store, fused", envelope=True, max_flagged=1.0)
    g.set_traversal(vr.SORT_LAST)
    out = torch.empty((H, W, 4), dtype=torch.float32, device="cuda")
    for call in (lambda: g.render(*views[0], W, H, 0.5, vr.MIP, out),
                 lambda: g.render(*views[0], W, H, 0.5, vr.ALPHA, out),        # steps outside [0.9, 1] need the float32 store (R20)
                 lambda: g.render(*views[0], W, H, 1.63, vr.ALPHA, out),
                 lambda: g.render(*views[0], W, H, vr.STEP_AUTO, vr.ALPHA, out),
                 lambda: g.upload(torch.from_numpy(data).cuda()),
                 lambda: g.download(np.empty((4, 4, 4), dtype=np.float32)),
                 lambda: g.debug_brick_data(0),
                 lambda: g.set_sampler(vr.SAMPLER_MANUAL),
                 lambda: g.release_store()):
        with pytest.raises(vr.VrError) as e:
            call()
        assert e.value.status == 4
    g.set_transfer_function(synth.tf_threshold(), synth.TF_VMIN, synth.TF_VMAX)
    with pytest.raises(vr.VrError):
        g.render(*views[0], W, H, 1.0, vr.ALPHA, out)                 # a stepped table needs the float32 store
    g.set_transfer_function(synth.tf_ramp(), synth.TF_VMIN, synth.TF_VMAX)
    assert np.abs(gpu_frame(g, *views[0], W, H, 1.0, vr.ALPHA) - before[0]).max() < 1e-3
    plain = vr.Volume(32, 32, 32, 16, 1)
    plain.upload(np.zeros((32, 32, 32), dtype=np.float32))
    with pytest.raises(vr.VrError):
        plain.release_store()


def _mip_both_samplers(vr, g, view, proj, W, H, step, pix, tex_sampler):
    """MIP frame, sub-images at `pix` and sample count with the hand-rolled sampler and through the arrays."""
    out = []
    for s in (vr.SAMPLER_MANUAL, tex_sampler):
        g.set_sampler(s)
        img = gpu_frame(g, view, proj, W, H, step, vr.MIP)
        out.append((img, g.debug_subimages(pix), g.debug_stats()["samples"]))
    return out


@pytest.mark.parametrize("texels", ["float32", "float16", "byte"])
@pytest.mark.parametrize("case", ["noise", "checkerboard", "outlier", "constant", "offset", "tiny", "tinier", "blanked", "ghost0", "ghost2"])
def test_mip_through_the_arrays_is_exact(vr, case, texels):
    """VR_MIP with the texture sampler: the filtered fetch only decides which samples CAN be the maximum (bound: range / 64
    of the brick); those are evaluated by the hand-rolled float32 sampler. The frame, every brick's scalar sub-image and
    the sample count must equal the hand-rolled path's bit for bit - also where the bound is tight (a checkerboard: cells
    span the brick's range), useless (one huge voxel), zero (constant data), dominated by rounding (a small range on a
    large offset) or not applicable (blanked bricks)."""
    rng = np.random.default_rng(5)
    cube = synth.Cube(19, 100, 90, 70, 10)
    data = cube.fill_host()
    ghost = {"ghost0": 0, "ghost2": 2}.get(case, 1)
    if case == "checkerboard":
        z, y, x = np.indices(data.shape)
        data = (((x + y + z) & 1) * 2.0 - 1.0).astype(np.float32) * rng.uniform(0.5, 8.0, size=data.shape).astype(np.float32)
    elif case == "outlier":
        data[33, 41, 57] = 3.0e6
    elif case == "constant":
        data[:] = 2.5
        data[:, :, 64:] = -1.0   # two constant halves: bricks with range 0 and bricks with a step
    elif case == "offset":
        data = (data * 1e-3 - 4000.0).astype(np.float32)  # range 0.02 at magnitude 4000: float32 rounding of the filters shows
    elif case == "tiny":
        data = (data * 1e-6).astype(np.float32)  # float16 subnormals (below 6e-5): texels keep 2^-25 absolute, not 2^-11 relative
    elif case == "tinier":
        data = (np.abs(data) * 2e-8).astype(np.float32)  # a brick's whole range inside ONE step (6e-8) of float16's subnormal grid
    elif case == "blanked":
        data[10:30, 5:25, 20:50] = np.nan
        data[3, 7, 60] = np.nan
    if case == "outlier" and texels == "float16":
        data[60, 20, 10] = -7.0e4  # beyond float16: that brick keeps the hand-rolled loop
    tex_sampler = {"float32": vr.SAMPLER_TEXTURE, "float16": vr.SAMPLER_TEXTURE_HALF, "byte": vr.SAMPLER_TEXTURE_BYTE}[texels]
    g, o = make_pair(cube, 32, ghost, data=data)
    W, H = 203, 117
    fr = synth.Framing(cube.nx, cube.ny, cube.nz, W, H)
    pix = seeded_pixels(9, W, H, 400)
    g.set_counting(1)
    for k, ortho, step in ((0, False, 0.5), (1, True, 0.5), (2, False, 1.0)):
        view, proj = fr.seeded(31, k), fr.proj(ortho)
        (m_img, m_sub, m_n), (t_img, t_sub, t_n) = _mip_both_samplers(vr, g, view, proj, W, H, step, pix, tex_sampler)
        assert np.array_equal(m_img, t_img, equal_nan=True), "%s view %d: frames differ by %g" % (case, k, np.nanmax(np.abs(m_img - t_img)))
        # a ray may stop once its maximum saturates the colour map (vmax): beyond that the scalar is not unique
        assert np.array_equal(np.minimum(m_sub, synth.TF_VMAX), np.minimum(t_sub, synth.TF_VMAX), equal_nan=True), \
            "%s view %d: sub-images differ" % (case, k)
        if np.nanmax(data) < synth.TF_VMAX:
            assert m_n == t_n   # no ray stops early: the same samples
        else:
            assert t_n >= m_n   # a saturated ray is noticed when its queue is emptied, a few samples later
        if k == 0 and case in ("noise", "checkerboard", "blanked"):
            check_mip(t_img, o.render(view, proj, W, H, step, oracle.MIP), "%s through the arrays" % case)


def test_narrow_arrays_serve_mip_only_and_switching_replaces_them(vr):
    """SAMPLER_TEXTURE_HALF / _BYTE: ALPHA frames keep the hand-rolled sampler bit for bit; switching samplers replaces the arrays."""
    import torch
    cube = synth.Cube(23, 96, 80, 64, 8)
    g, o = make_pair(cube, 32, 1)
    W, H = 160, 100
    fr = synth.Framing(cube.nx, cube.ny, cube.nz, W, H)
    view, proj = fr.seeded(5, 1), fr.proj(False)
    a_man = gpu_frame(g, view, proj, W, H, 0.5, vr.ALPHA)
    m_man = gpu_frame(g, view, proj, W, H, 0.5, vr.MIP)
    for s in (vr.SAMPLER_TEXTURE_HALF, vr.SAMPLER_TEXTURE, vr.SAMPLER_TEXTURE_BYTE, vr.SAMPLER_TEXTURE_HALF, vr.SAMPLER_MANUAL,
              vr.SAMPLER_TEXTURE_BYTE):
        g.set_sampler(s)
        assert np.array_equal(gpu_frame(g, view, proj, W, H, 0.5, vr.MIP), m_man)
        a = gpu_frame(g, view, proj, W, H, 0.5, vr.ALPHA)
        if s in (vr.SAMPLER_TEXTURE, vr.SAMPLER_TEXTURE_HALF):
            assert 1e-7 < np.abs(a - a_man).max() < 0.02  # the arrays' filtered values
        else:
            assert np.array_equal(a, a_man)
    # R22's guard: data whose magnitude is large against the table's range is too coarse in float16 - ALPHA frames then
    # come from the hand-rolled sampler (bit for bit) although the float16 arrays are in force; MIP stays exact either way
    far = vr.Volume(cube.nx, cube.ny, cube.nz, 32, 1)
    shifted = (cube.fill_host() + 300.0).astype(np.float32)
    far.upload(shifted)
    far.set_transfer_function(synth.tf_ramp(), synth.TF_VMIN + 300.0, synth.TF_VMAX + 300.0)
    a_far, m_far = gpu_frame(far, view, proj, W, H, 0.5, vr.ALPHA), gpu_frame(far, view, proj, W, H, 0.5, vr.MIP)
    far.set_sampler(vr.SAMPLER_TEXTURE_HALF)
    assert np.array_equal(gpu_frame(far, view, proj, W, H, 0.5, vr.ALPHA), a_far)
    assert np.array_equal(gpu_frame(far, view, proj, W, H, 0.5, vr.MIP), m_far)
    far.set_sampler(vr.SAMPLER_TEXTURE)
    assert 1e-7 < np.abs(gpu_frame(far, view, proj, W, H, 0.5, vr.ALPHA) - a_far).max() < 0.02  # float32 texels do serve it
    far.close()
    # an upload is followed by the byte arrays too (their scale is the NEW range of each brick)
    d2 = cube.fill_host()
    d2[20:40, 30:50, 40:60] += 6.0
    g.upload(torch.from_numpy(d2).cuda())
    m_tex = gpu_frame(g, view, proj, W, H, 0.5, vr.MIP)
    g.set_sampler(vr.SAMPLER_MANUAL)
    m2 = gpu_frame(g, view, proj, W, H, 0.5, vr.MIP)
    assert np.array_equal(m_tex, m2) and np.abs(m2 - m_man).max() > 1e-2


@pytest.mark.parametrize("texels", ["float32", "float16", "byte"])
def test_filter_error_stays_inside_the_bound_the_mip_filter_relies_on(vr, texels):
    """R23's constant, measured where it is largest: a +-1 checkerboard (every cell spans the brick's whole range along
    every axis), noise, and noise on a large offset. The filtered fetch must stay within range / 64 (+ range / 500 for
    8-bit texels) + the magnitude term of the exact value, with room to spare."""
    sid = {"float32": vr.SAMPLER_TEXTURE, "float16": vr.SAMPLER_TEXTURE_HALF, "byte": vr.SAMPLER_TEXTURE_BYTE}[texels]
    range_eps = 1.0 / 64 + (1.0 / 500 if texels == "byte" else 0.0)
    mag_eps = {"float32": 2.0 ** -14, "float16": 2.0 ** -9, "byte": 2.0 ** -12}[texels]
    cube = synth.Cube(7, 96, 96, 96, 6)
    noise = cube.fill_host()
    z, y, x = np.indices(noise.shape)
    cases = {"checkerboard": (((x + y + z) & 1) * 2.0 - 1.0).astype(np.float32), "noise": noise,
             "offset noise": (noise + 300.0).astype(np.float32)}
    for name, data in cases.items():
        g = vr.Volume(96, 96, 96, 32, 1)
        g.upload(data)
        g.set_sampler(sid)
        worst = 0.0
        for b in (0, 13, 26):
            err, rng = g.debug_tex_error(b, 1 << 21, seed=b + 1)
            mag = float(np.abs(data).max())
            bound = rng * range_eps + mag * mag_eps
            assert rng > 0 and err <= 0.85 * bound, (name, texels, b, err, rng, bound)
            worst = max(worst, err / rng)
        print("filter error / range, %s texels, %s: %.5f (bound %.5f)" % (texels, name, worst, range_eps))
        g.close()


@pytest.mark.parametrize("case", range(int(__import__("os").environ.get("VR_SCALE_CASES", "24"))))
def test_mip_exactness_over_scales_and_offsets(vr, case):
    """R23 across magnitudes: the same noise cube scaled by 10^-12 .. 10^6 and shifted by up to 10^4 ranges (float16
    subnormals and overflow, 8-bit steps far above the data's own spread, float32 rounding of the decode): MIP frames
    through every texel width equal the hand-rolled frame."""
    rng = np.random.default_rng(4000 + case)
    dims = tuple(int(v) for v in rng.integers(24, 60, 3))
    base = synth.Cube(900 + case, *dims, 3).fill_host()
    scale = 10.0 ** rng.uniform(-12, 6)
    offset = scale * float(rng.choice([0.0, 0.0, 1.0, -30.0, 1e3, -1e4]))
    data = (base * scale + offset).astype(np.float32)
    if rng.random() < 0.3:
        data[tuple(int(v) for v in rng.integers(0, 20, 3))] = np.float32(scale * 1e4)  # one voxel far outside
    brick = int(rng.choice([8, 16, 32]))
    g = vr.Volume(*dims, brick, int(rng.choice([0, 1, 2])))
    g.upload(data)
    lo, hi = float(np.min(data)), float(np.max(data))
    g.set_transfer_function(synth.tf_ramp(), lo, hi if hi > lo else lo + 1.0)
    W, H = 96, 80
    fr = synth.Framing(*dims, W, H)
    view, proj = fr.seeded(50 + case, case), fr.proj(bool(case & 1))
    step = float(rng.choice([0.5, 1.0, 0.37]))
    want = gpu_frame(g, view, proj, W, H, step, vr.MIP)
    for s in (vr.SAMPLER_TEXTURE, vr.SAMPLER_TEXTURE_HALF, vr.SAMPLER_TEXTURE_BYTE):
        g.set_sampler(s)
        got = gpu_frame(g, view, proj, W, H, step, vr.MIP)
        assert np.array_equal(got, want), (case, s, scale, offset, float(np.abs(got - want).max()))


def test_nearly_opaque_samples_at_small_steps_are_taken_by_hand(vr):
    """R20's guard. With steps below one voxel the opacity correction 1 - (1 - a)^w has an unbounded slope where the table's
    opacity nears 1: a source whose peak sits just around the top of the table (a -> 1) turned the filter's 1e-3 value error
    into 7e-3 of the pixel (randomised case 1082). Such samples are re-evaluated by the hand-rolled sampler."""
    dims = (40, 36, 32)
    z, y, x = np.indices(dims[::-1]).astype(np.float32)
    r2 = (x - 20.3) ** 2 + (y - 17.6) ** 2 + (z - 15.2) ** 2
    data = (np.random.default_rng(3).normal(0, 0.3, dims[::-1]) + 10.9 * np.exp(-r2 / (2 * 2.2 ** 2))).astype(np.float32)  # peak just above vmax = 10
    W, H = 120, 100
    fr = synth.Framing(*dims, W, H)
    for texels in TEXELS:
        for tau in (0.9, 0.99, 2.0):
            g, o = tex_pair(vr, synth.Cube(1, *dims, 1), 16, 1, tf=synth.tf_ramp(), tau=tau, data=data, texels=texels)
            o.set_ert_margin(0.02 * (1.0 - tau) if tau < 1 else 2e-4)
            for k, step in ((0, 0.5), (1, 0.37), (2, 0.25)):
                view, proj = fr.seeded(9, k), fr.proj(False)
                check_alpha(gpu_frame(g, view, proj, W, H, step, vr.ALPHA), o.render(view, proj, W, H, step, oracle.ALPHA), tau,
                            "peak at the table's top, %s, tau %g, step %g" % (texels, tau, step), envelope=True, max_flagged=1.0)


@pytest.mark.parametrize("case", range(int(__import__("os").environ.get("VR_RELEASE_CASES", "16"))))
def test_randomised_released_stores(vr, case):
    """Seeded random volumes on VR_LAYOUT_TILED_RELEASABLE handles, released to float32 or float16 arrays: both traversals
    against the oracle (steps in [0.9, 1]: what a released store renders), blanked bricks keep their float32 cells."""
    import torch
    rng = np.random.default_rng(7000 + case)
    dims = tuple(int(v) for v in rng.integers(20, 80, 3))
    brick = int(rng.choice([8, 16, 32]))
    ghost = int(rng.choice([1, 1, 2]))
    data = synth.Cube(300 + case, *dims, int(rng.integers(1, 8))).fill_host()
    if rng.random() < 0.4:
        data[rng.random(data.shape) < 0.005] = np.nan
    tf = [synth.tf_ramp, synth.tf_translucent][int(rng.integers(0, 2))]()
    tau = float(rng.choice([0.99, 0.9, 2.0]))
    step = float(rng.choice([1.0, 1.0, 0.9, 0.95]))
    half = bool(rng.integers(0, 2))
    W, H = int(rng.integers(40, 130)), int(rng.integers(30, 100))
    fr = synth.Framing(*dims, W, H)
    view, proj = fr.seeded(800 + case, case), fr.proj(bool(rng.integers(0, 2)))
    g = vr.Volume(*dims, brick, ghost, layout=vr.LAYOUT_TILED_RELEASABLE)
    g.upload(torch.from_numpy(data).cuda())
    o = oracle.Volume(*dims, brick, ghost, data=data)
    one = oracle.Volume(*dims, 128, 1, data=data)
    for v in (g, o, one):
        v.set_transfer_function(tf, synth.TF_VMIN, synth.TF_VMAX)
        v.set_early_termination(tau)
    band = 0.02 * (1.0 - tau) if tau < 1.0 else 2e-4
    o.set_ert_margin(band)
    one.set_ert_margin(band)
    if half:
        g.set_sampler(vr.SAMPLER_TEXTURE_HALF)
    assert g.release_store() >= 0
    for trav, orc in ((vr.SORT_LAST, o), (vr.FUSED, one)):
        g.set_traversal(trav)
        check_alpha(gpu_frame(g, view, proj, W, H, step, vr.ALPHA), orc.render(view, proj, W, H, step, oracle.ALPHA), tau,
                    "released case %d (%s texels, traversal %d)" % (case, "float16" if half else "float32", trav), envelope=True,
                    max_flagged=1.0)
    g.close()


def test_tables_steeper_than_a_full_range_ramp_keep_the_hand_rolled_sampler(vr):
    """R20 (ii): the frame's error through the arrays grows with the table's slope (2.7e-3 at 1.5 times the ramp's), so
    only tables no steeper than a ramp over the whole range take their values from the arrays; a ramp over the top half of
    the range renders exactly as with the hand-rolled sampler although the texture sampler is in force."""
    c = synth.CONFIGS["c0"]
    cube = synth.config_cube("c0")
    W, H = 128, 128
    fr = synth.Framing(cube.nx, cube.ny, cube.nz, W, H)
    view, proj = fr.seeded(77, 0), fr.proj(False)
    for slope, through_arrays in ((1.0, True), (1.05, True), (1.5, False), (2.0, False)):
        tf = synth.tf_ramp()
        n = tf.shape[0]
        u = np.arange(n) / (n - 1)
        tf[:, 3] = np.clip((u - (1 - 1 / slope)) * slope, 0, 1).astype(np.float32)
        g, o = make_pair(cube, c["brick"], 1, tf=tf, tau=0.99)
        o.set_ert_margin(2e-4)
        man = gpu_frame(g, view, proj, W, H, 0.5, vr.ALPHA)
        for s in (vr.SAMPLER_TEXTURE, vr.SAMPLER_TEXTURE_HALF):
            g.set_sampler(s)
            img = gpu_frame(g, view, proj, W, H, 0.5, vr.ALPHA)
            assert (not np.array_equal(img, man)) == through_arrays, (slope, s)
            check_alpha(img, o.render(view, proj, W, H, 0.5, oracle.ALPHA), 0.99, "slope %g" % slope, envelope=True, max_flagged=1.0)


def test_data_too_rough_for_the_table_keeps_the_hand_rolled_sampler(vr):
    """R20 (vii): the filter's error scales with the voxel-to-voxel differences against the table's range. The same cube
    three times as noisy under the same table (or the same cube under a table a third as wide) fails the guard and renders
    exactly as with the hand-rolled sampler; the benchmark statistics pass it."""
    c = synth.CONFIGS["c0"]
    cube = synth.config_cube("c0")
    data = cube.fill_host()
    W, H = 128, 128
    fr = synth.Framing(cube.nx, cube.ny, cube.nz, W, H)
    view, proj = fr.seeded(77, 1), fr.proj(False)
    for scale, lo, hi, through_arrays in ((1.0, synth.TF_VMIN, synth.TF_VMAX, True), (3.0, synth.TF_VMIN, synth.TF_VMAX, False),
                                         (1.0, -1.0, 3.3, False), (0.3, synth.TF_VMIN, synth.TF_VMAX, True)):
        d = (data * scale).astype(np.float32)
        g = vr.Volume(cube.nx, cube.ny, cube.nz, c["brick"], 1)
        g.upload(d)
        o = oracle.Volume(cube.nx, cube.ny, cube.nz, c["brick"], 1, data=d)
        for v in (g, o):
            v.set_transfer_function(synth.tf_ramp(), lo, hi)
            v.set_early_termination(0.99)
        o.set_ert_margin(2e-4)
        rng_, slope, ok = g.debug_tex_alpha_guard()
        assert ok == through_arrays and abs(slope - 1.004) < 1e-3, (scale, lo, hi, rng_, slope, ok)
        man = gpu_frame(g, view, proj, W, H, 0.5, vr.ALPHA)
        g.set_sampler(vr.SAMPLER_TEXTURE)
        img = gpu_frame(g, view, proj, W, H, 0.5, vr.ALPHA)
        assert (not np.array_equal(img, man)) == through_arrays
        check_alpha(img, o.render(view, proj, W, H, 0.5, oracle.ALPHA), 0.99, "roughness guard", envelope=True, max_flagged=1.0)
