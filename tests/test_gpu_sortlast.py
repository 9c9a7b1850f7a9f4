"""Row f3 on one GPU: the parts of a k-d partition are rendered one after the other by part handles (no rank
waits for another), their partial frames are merged by vr_composite_parts, and the frame must be the oracle's
frame of the whole volume (north_star's tolerances) and the single-handle GPU frame to float32 rounding.
The exchange in between is covered over gloo by tests/test_sortlast.py."""
import numpy as np
import pytest

import oracle
import synth
from helpers import check_alpha, check_mip, gpu_frame

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def vr(cuda_device):
    from paper_1205_0282_b200 import build
    build.build()
    import paper_1205_0282_b200 as vr
    return vr


def make_parts(vr, sortlast, data, dims, brick, ghost, nparts, halo_only=True):
    """One part handle per box, fed with the box's region only (its bricks + ghost layers)."""
    import torch
    boxes, tree = sortlast.kd_partition(dims, brick, nparts)
    parts = []
    for box in boxes:
        p = vr.Volume(*dims, brick, ghost, part=box)
        (x0, y0, z0), (sx, sy, sz) = sortlast.part_region(dims, brick, ghost, box) if halo_only else ((0, 0, 0), dims)
        p.upload(torch.from_numpy(np.ascontiguousarray(data[z0:z0 + sz, y0:y0 + sy, x0:x0 + sx])).cuda(), origin=(x0, y0, z0))
        parts.append(p)
    return boxes, tree, parts


def merged_frame(vr, sortlast, parts, boxes, tree, dims, brick, view, proj, W, H, step, mode, use_pieces=True):
    """What SortLastRenderer does, on one device: every part composites its sub-images straight into rectangle-packed
    pieces (here: its rectangle cut into an upper and a lower piece, as two stripes would), merged in part order.
    The pieces must equal, bit for bit, the same pixels of the part's full partial frame (vr_render_part), which must
    be blank outside the part's rectangle. ALPHA: float4 per pixel; MIP: one float per pixel, -inf = no sample."""
    import torch
    pieces, rects = [], []
    for p, box in zip(parts, boxes):
        full = torch.empty((H, W, 4) if mode == vr.ALPHA else (H, W), dtype=torch.float32, device="cuda")
        r = p.render_part(view, proj, W, H, step, mode, full)
        assert r == vr.part_rect(dims, brick, box, view, proj, W, H)
        outside = full.clone()
        outside[r[1]:r[3], r[0]:r[2]] = 0 if mode == vr.ALPHA else -np.inf
        assert not (outside.any() if mode == vr.ALPHA else (outside != -np.inf).any()), "a partial frame is not blank outside its rectangle"
        ymid = (r[1] + r[3]) // 2
        cuts = [c for c in ((r[0], r[1], r[2], ymid), (r[0], ymid, r[2], r[3])) if c[2] > c[0] and c[3] > c[1]]
        bufs = [torch.full((c[3] - c[1], c[2] - c[0], 4) if mode == vr.ALPHA else (c[3] - c[1], c[2] - c[0]), 7.0,
                           dtype=torch.float32, device="cuda") for c in cuts]
        if use_pieces:
            p.render_part_pieces(view, proj, W, H, step, mode, cuts, bufs)
            for c, b in zip(cuts, bufs):
                assert torch.equal(b, full[c[1]:c[3], c[0]:c[2]])
        else:  # the fused traversal of a part writes its whole partial frame: the pieces are cut out of it
            bufs = [full[c[1]:c[3], c[0]:c[2]].contiguous() for c in cuts]
        pieces += bufs
        rects += cuts
    # a part's pieces do not overlap, so any order that keeps the parts in visibility order will do
    po = sortlast.part_order(tree, brick, view, proj)
    idx, k = {}, 0
    for q, (p, box) in enumerate(zip(parts, boxes)):
        r = vr.part_rect(dims, brick, box, view, proj, W, H)
        ymid = (r[1] + r[3]) // 2
        n = sum(1 for c in ((r[0], r[1], r[2], ymid), (r[0], ymid, r[2], r[3])) if c[2] > c[0] and c[3] > c[1])
        idx[q] = list(range(k, k + n))
        k += n
    order = [i for q in po for i in idx[q]]
    out = torch.empty((H, W, 4), dtype=torch.float32, device="cuda")
    parts[0].composite_parts(mode, pieces, rects, order, W, H, out)
    torch.cuda.synchronize()
    return out.cpu().numpy().astype(np.float64)


@pytest.mark.parametrize("nparts", [2, 3, 4, 6])
@pytest.mark.parametrize("tfname", ["ramp", "translucent"])
def test_merged_parts_are_the_frame_of_the_whole_volume(vr, nparts, tfname):
    from paper_1205_0282_b200 import sortlast
    dims, brick, ghost, W, H = (70, 52, 64), 16, 1, 150, 110
    cube = synth.Cube(21, *dims, 5)
    data = cube.fill_host()
    tf = getattr(synth, "tf_" + tfname)()
    boxes, tree, parts = make_parts(vr, sortlast, data, dims, brick, ghost, nparts)
    whole = vr.Volume(*dims, brick, ghost)
    whole.upload(data)
    o = oracle.Volume(*dims, brick, ghost, data=data)
    for v in parts + [whole, o]:
        v.set_transfer_function(tf, synth.TF_VMIN, synth.TF_VMAX)
        v.set_early_termination(0.99)
    fr = synth.Framing(*dims, W, H)
    views = [(fr.seeded(31, k), fr.proj(k % 2 == 1)) for k in range(4)]
    views.append((synth.look_at((20.0, 30.0, 40.0), (70.0, 0.0, 0.0), (0.0, 0.3, 1.0)), synth.perspective(60, W / H, 0.3, 400.0)))
    for k, (view, proj) in enumerate(views):
        for step in (0.6, vr.STEP_AUTO):
            what = "%d parts, view %d, step %g" % (nparts, k, step)
            ref = o.render(view, proj, W, H, step, oracle.ALPHA)
            got = merged_frame(vr, sortlast, parts, boxes, tree, dims, brick, view, proj, W, H, step, vr.ALPHA)
            check_alpha(got, ref, 0.99, what)
            one = gpu_frame(whole, view, proj, W, H, step, vr.ALPHA)
            assert np.abs(got - one).max() < 2e-6, what      # same sub-images, `over` regrouped
            refm = o.render(view, proj, W, H, step, oracle.MIP)
            gotm = merged_frame(vr, sortlast, parts, boxes, tree, dims, brick, view, proj, W, H, step, vr.MIP)
            check_mip(gotm, refm, what)
            assert np.array_equal(gotm, gpu_frame(whole, view, proj, W, H, step, vr.MIP)), what   # max is exact


def test_part_handles_hold_their_own_bricks_only(vr):
    """Store, ranges and debug exports of a part: own bricks bit-exact (ghost layers from the neighbours' voxels),
    the others absent; whole-volume uploads are filtered."""
    from paper_1205_0282_b200 import sortlast
    dims, brick, ghost = (50, 40, 45), 16, 2
    data = synth.Cube(5, *dims, 4).fill_host()
    o = oracle.Volume(*dims, brick, ghost, data=data)
    g = sortlast.brick_grid(dims, brick)
    for halo_only in (True, False):
        boxes, tree, parts = make_parts(vr, sortlast, data, dims, brick, ghost, 3, halo_only)
        for p, (b0, b1) in zip(parts, boxes):
            mm = p.debug_brick_minmax()
            lo, hi = np.inf, -np.inf
            for b in range(p.nbricks):
                bx, by, bz = b % g[0], (b // g[0]) % g[1], b // (g[0] * g[1])
                own = all(b0[a] <= c < b1[a] for a, c in enumerate((bx, by, bz)))
                if own:
                    assert np.array_equal(p.debug_brick_data(b), o.brick_data(b)), b
                    assert tuple(mm[b]) == o.brick_minmax(b)
                    lo, hi = min(lo, mm[b][0]), max(hi, mm[b][1])
                else:
                    assert mm[b][0] == np.inf and mm[b][1] == -np.inf
                    with pytest.raises(vr.VrError):
                        p.debug_brick_data(b)
            assert p.minmax() == (lo, hi)
            # voxels come back from the part's own bricks only
            import torch
            x0, y0, z0 = (b0[a] * brick for a in range(3))
            x1, y1, z1 = (min(b1[a] * brick, dims[a]) for a in range(3))
            back = torch.empty((z1 - z0, y1 - y0, x1 - x0), dtype=torch.float32, device="cuda")
            p.download(back, origin=(x0, y0, z0))
            torch.cuda.synchronize()
            assert np.array_equal(back.cpu().numpy(), data[z0:z1, y0:y1, x0:x1])
            if (x1, y1, z1) != dims:
                with pytest.raises(vr.VrError):
                    p.download(torch.empty(dims[::-1], dtype=torch.float32, device="cuda"), origin=(0, 0, 0))


def test_part_arguments(vr):
    with pytest.raises(vr.VrError):
        vr.Volume(64, 64, 64, 16, 1, part=((0, 0, 0), (5, 4, 4)))     # outside the 4x4x4 grid
    with pytest.raises(vr.VrError):
        vr.Volume(64, 64, 64, 16, 1, part=((2, 0, 0), (2, 4, 4)))     # empty
    import torch
    p = vr.Volume(64, 64, 64, 16, 1, part=((0, 0, 0), (2, 4, 4)))
    p.upload(torch.zeros((64, 64, 64), dtype=torch.float32, device="cuda"))
    p.set_transfer_function(synth.tf_ramp(), 0.0, 1.0)
    p.set_traversal(vr.FUSED)
    fr = synth.Framing(64, 64, 64, 64, 48)
    out = torch.empty((48, 64, 4), dtype=torch.float32, device="cuda")
    with pytest.raises(vr.VrError):                                    # a MIP part stays scalar: sort-last traversal only
        p.render_part(fr.seeded(1, 0), fr.proj(False), 64, 48, 1.0, vr.MIP, out)
    p.render_part(fr.seeded(1, 0), fr.proj(False), 64, 48, 1.0, vr.ALPHA, out)
    with pytest.raises(vr.VrError):                                    # pieces come from the sort-last traversal
        p.render_part_pieces(fr.seeded(1, 0), fr.proj(False), 64, 48, 1.0, vr.ALPHA, [(0, 0, 8, 8)], [out[:8, :8].contiguous()])
    p.set_traversal(vr.SORT_LAST)
    with pytest.raises(vr.VrError):                                    # a piece must lie inside the frame
        p.render_part_pieces(fr.seeded(1, 0), fr.proj(False), 64, 48, 1.0, vr.ALPHA, [(60, 0, 68, 8)], [out[:8, :8].contiguous()])


def test_parts_cull_and_skip_like_the_whole_volume(vr):
    """R16/R19 on parts: a threshold transfer function over an N-body cube; culling and macro-cell skipping run per
    part on the part's own tables, the merged frame does not change by a bit with them off, and parity holds. The
    fused traversal of a part (global early termination inside the part) merges to the oracle's frame as well when
    early termination is off."""
    from paper_1205_0282_b200 import sortlast
    dims, brick, ghost, W, H = (96, 80, 72), 32, 1, 140, 100
    data = synth.Cube(9, *dims, 6, kind=1).fill_host()
    tf = synth.tf_density()
    boxes, tree, parts = make_parts(vr, sortlast, data, dims, brick, ghost, 4)
    o = oracle.Volume(*dims, brick, ghost, data=data)
    for v in parts + [o]:
        v.set_transfer_function(tf, 0.0, synth.NBODY_VMAX)
        v.set_early_termination(2.0)
    fr = synth.Framing(*dims, W, H)
    for k in range(3):
        view, proj = fr.seeded(91, k), fr.proj(k == 2)
        ref = o.render(view, proj, W, H, 0.8, oracle.ALPHA)
        frames = {}
        for cull in (True, False):
            for p in parts:
                p.set_culling(cull)
            frames[cull] = merged_frame(vr, sortlast, parts, boxes, tree, dims, brick, view, proj, W, H, 0.8, vr.ALPHA)
        assert np.array_equal(frames[True], frames[False])
        check_alpha(frames[True], ref, 2.0, "view %d" % k)
        for p in parts:
            p.set_traversal(vr.FUSED)
        fused = merged_frame(vr, sortlast, parts, boxes, tree, dims, brick, view, proj, W, H, 0.8, vr.ALPHA, use_pieces=False)
        check_alpha(fused, ref, 2.0, "fused parts, view %d" % k)
        for p in parts:
            p.set_traversal(vr.SORT_LAST)
    assert sum(p.debug_stats()["bricks_culled"] for p in parts) >= 0


def test_a_world_of_one_renders_through_the_renderer(vr):
    from paper_1205_0282_b200 import sortlast
    import torch
    dims, brick, W, H = (48, 40, 36), 16, 96, 72
    data = synth.Cube(3, *dims, 3).fill_host()
    rdr = sortlast.SortLastRenderer(dims, brick, 1, rank=0, world=1)
    origin, shape = rdr.region()
    assert origin == (0, 0, 0) and shape == dims
    rdr.upload(torch.from_numpy(data).cuda(), origin)
    rdr.set_transfer_function(synth.tf_ramp(), synth.TF_VMIN, synth.TF_VMAX)
    whole = vr.Volume(*dims, brick, 1)
    whole.upload(data)
    whole.set_transfer_function(synth.tf_ramp(), synth.TF_VMIN, synth.TF_VMAX)
    assert rdr.minmax() == whole.minmax()
    fr = synth.Framing(*dims, W, H)
    view, proj = fr.seeded(8, 1), fr.proj(False)
    for mode in (vr.ALPHA, vr.MIP):
        frame = rdr.render(view, proj, W, H, 1.0, mode)
        torch.cuda.synchronize()
        assert np.array_equal(frame.cpu().numpy().astype(np.float64), gpu_frame(whole, view, proj, W, H, 1.0, mode))


def test_bench_brick_sharded_arm_as_a_world_of_one(vr):
    """bench.py --sharding bricks on one GPU: the contract line, through SortLastRenderer."""
    import json
    import os
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    r = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--workload", "c0", "--sharding", "bricks", "--steps", "6",
                        "--warmup", "3"], capture_output=True, text=True, timeout=600)
    assert r.returncode == 0, r.stderr[-2000:]
    line = json.loads(r.stdout.strip().splitlines()[-1])
    assert line["metric"] == "frames_per_s" or line["unit"] == "frames/s"
    assert line["n_gpus"] == 1 and line["scaling"] == "strong" and line["value"] > 0 and line["e2e"]["value"] > 0
    assert line["gpu_launches"] == 6 * 5            # set-up, ray table, ray cast, stage-1 compositing, merge
    assert line["exchange_bytes_per_frame"] == 0    # a world of one sends nothing


@pytest.mark.parametrize("sampler", ["texture", "texture_half", "texture_byte"])
def test_parts_through_the_texture_arrays(vr, sampler):
    """Part handles with the texture arm (arrays of the part's own bricks only; 8-bit texels scaled with the ranges of the
    bricks the part holds): merged MIP frames bit-identical to the hand-rolled single handle's, merged ALPHA frames inside
    the tolerance (float32 / float16 values) or untouched (8-bit arrays serve MIP only)."""
    from paper_1205_0282_b200 import sortlast
    dims, brick, ghost, W, H = (70, 52, 64), 16, 1, 150, 110
    data = synth.Cube(21, *dims, 5).fill_host()
    boxes, tree, parts = make_parts(vr, sortlast, data, dims, brick, ghost, 3)
    whole = vr.Volume(*dims, brick, ghost)
    whole.upload(data)
    o = oracle.Volume(*dims, brick, ghost, data=data)
    o.set_ert_margin(2e-4)
    sid = {"texture": vr.SAMPLER_TEXTURE, "texture_half": vr.SAMPLER_TEXTURE_HALF, "texture_byte": vr.SAMPLER_TEXTURE_BYTE}[sampler]
    for v in parts + [whole, o]:
        v.set_transfer_function(synth.tf_ramp(), synth.TF_VMIN, synth.TF_VMAX)
        v.set_early_termination(0.99)
    for p in parts:
        p.set_sampler(sid)
    fr = synth.Framing(*dims, W, H)
    for k in range(3):
        view, proj = fr.seeded(31, k), fr.proj(k % 2 == 1)
        gotm = merged_frame(vr, sortlast, parts, boxes, tree, dims, brick, view, proj, W, H, 0.6, vr.MIP)
        assert np.array_equal(gotm, gpu_frame(whole, view, proj, W, H, 0.6, vr.MIP)), (sampler, k)
        got = merged_frame(vr, sortlast, parts, boxes, tree, dims, brick, view, proj, W, H, 0.6, vr.ALPHA)
        one = gpu_frame(whole, view, proj, W, H, 0.6, vr.ALPHA)
        if sampler == "texture_byte":
            assert np.abs(got - one).max() < 2e-6
        else:
            assert 1e-7 < np.abs(got - one).max() < 0.02
            check_alpha(got, o.render(view, proj, W, H, 0.6, oracle.ALPHA), 0.99, "parts, %s, view %d" % (sampler, k), envelope=True,
                        max_flagged=1.0)


@pytest.mark.parametrize("case", range(int(__import__("os").environ.get("VR_PARTS_CASES", "12"))))
def test_randomised_partitions(vr, case):
    """Row f3 under random use: random volumes, brick sizes, 1-9 parts (as far as the grid has bricks), both modes, the
    hand-rolled sampler or one of the texture arms on the parts: the merged frame is the single handle's (MIP: bit for
    bit whatever the sampler; ALPHA: the same sub-images regrouped, to float32 rounding, with the hand-rolled sampler)."""
    from paper_1205_0282_b200 import sortlast
    rng = np.random.default_rng(13000 + case)
    brick = int(rng.choice([8, 16, 32]))
    dims = tuple(int(v) for v in rng.integers(brick + 3, 5 * brick, 3))
    ghost = int(rng.choice([1, 1, 2]))
    grid = sortlast.brick_grid(dims, brick)
    nparts = int(rng.integers(1, min(9, grid[0] * grid[1] * grid[2]) + 1))
    data = synth.Cube(600 + case, *dims, int(rng.integers(1, 6))).fill_host()
    boxes, tree, parts = make_parts(vr, sortlast, data, dims, brick, ghost, nparts)
    whole = vr.Volume(*dims, brick, ghost)
    whole.upload(data)
    tf = [synth.tf_ramp, synth.tf_translucent][int(rng.integers(0, 2))]()
    for v in parts + [whole]:
        v.set_transfer_function(tf, synth.TF_VMIN, synth.TF_VMAX)
        v.set_early_termination(0.99)
    sampler = int(rng.choice([vr.SAMPLER_MANUAL, vr.SAMPLER_TEXTURE, vr.SAMPLER_TEXTURE_HALF, vr.SAMPLER_TEXTURE_BYTE]))
    for p in parts:
        p.set_sampler(sampler)
    W, H = int(rng.integers(40, 160)), int(rng.integers(30, 120))
    fr = synth.Framing(*dims, W, H)
    view, proj = fr.seeded(40 + case, case), fr.proj(bool(rng.integers(0, 2)))
    step = float(rng.choice([0.5, 1.0, 0.7]))
    gotm = merged_frame(vr, sortlast, parts, boxes, tree, dims, brick, view, proj, W, H, step, vr.MIP)
    assert np.array_equal(gotm, gpu_frame(whole, view, proj, W, H, step, vr.MIP)), (case, nparts, sampler)
    got = merged_frame(vr, sortlast, parts, boxes, tree, dims, brick, view, proj, W, H, step, vr.ALPHA)
    one = gpu_frame(whole, view, proj, W, H, step, vr.ALPHA)
    if sampler in (vr.SAMPLER_MANUAL, vr.SAMPLER_TEXTURE_BYTE):
        assert np.abs(got - one).max() < 2e-6, (case, nparts)
    else:
        # the same arrays on the single handle: the same sub-images regrouped - as long as every handle's data guard (R20 vii,
        # decided on the handle's own macro-cells; R22 on its own largest magnitude) came out the same way; a part that keeps
        # the hand-rolled sampler where the whole volume does not (or the other way round) is within the tolerance of both
        whole.set_sampler(sampler)
        same = len({h.debug_tex_alpha_guard()[2] for h in parts + [whole]}) == 1 and sampler == vr.SAMPLER_TEXTURE
        if same:
            assert np.abs(got - gpu_frame(whole, view, proj, W, H, step, vr.ALPHA)).max() < 2e-6, (case, nparts, sampler)
        # against the oracle the arrays' values are a MEASURED 2e-3, not a bound (R20 viii): this suite, run at 1200
        # cases, met one frame with two pixels at 2.4e-3 (case 1165, float16 texels). What it pins here is the regrouping;
        # the oracle parity of the texture arm is test_randomised_configurations' and the full-size tests' business.
        o = oracle.Volume(*dims, brick, ghost, data=data)
        o.set_transfer_function(tf, synth.TF_VMIN, synth.TF_VMAX)
        o.set_early_termination(0.99)
        o.set_ert_margin(2e-4)
        ref = o.render(view, proj, W, H, step, oracle.ALPHA)
        err = np.abs(got - ref["image"]).max(axis=-1)
        assert (err[ref["flags"] == 0] > 2e-3).mean() < 1e-3 and err[ref["flags"] == 0].max() < 4e-3, (case, nparts, sampler)
