"""Row f3 on CPUs: the k-d partition, the part visibility order, the part rectangles and the exchange protocol of
paper_1205_0282_b200.sortlast over gloo (world sizes 2 and 3), with the oracle standing in for the two kernels on
either side of the exchange (the GPU tests run the same protocol step by step with libvr's own)."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import oracle
import paper_1205_0282_b200 as vr
import synth
from paper_1205_0282_b200 import sortlast


from oracle import parts as oparts


# The partition and the part order exist twice: libvr's (vr_kd_partition / vr_part_order, C++, behind the C ABI: host
# arithmetic, callable without a GPU) and the oracle's plain statement (oracle/parts.py). The pins below run on BOTH;
# a last test demands that the two agree exactly.
def _nested(flat, t=0):
    axis, cut, lo, hi = (int(c) for c in flat[t])
    return ("leaf", cut) if axis < 0 else ("node", axis, cut, _nested(flat, lo), _nested(flat, hi))


class _Libvr:
    name = "libvr"

    @staticmethod
    def kd_partition(dims, brick, nparts):
        try:
            boxes, flat = sortlast.kd_partition(dims, brick, nparts)
        except vr.VrError as e:
            raise ValueError(str(e))
        return boxes, _nested(flat)

    @staticmethod
    def part_order(tree, brick, view, proj):
        return sortlast.part_order(oparts.flatten(tree), brick, view, proj)


class _Oracle:
    name = "oracle"
    kd_partition = staticmethod(oparts.kd_partition)
    part_order = staticmethod(oparts.part_order)


IMPLS = [_Oracle, _Libvr]


# --------------------------------------------------------------------------------- partition
@pytest.mark.parametrize("impl", IMPLS, ids=lambda i: i.name)
@pytest.mark.parametrize("dims,brick", [((64, 64, 64), 16), ((100, 37, 64), 16), ((33, 200, 90), 8), ((512, 512, 6400), 256)])
@pytest.mark.parametrize("nparts", [1, 2, 3, 4, 5, 6, 7, 8])
def test_kd_partition_tiles_the_brick_grid(impl, dims, brick, nparts):
    g = sortlast.brick_grid(dims, brick)
    boxes, tree = impl.kd_partition(dims, brick, nparts)
    owner = np.full(g[::-1], -1, dtype=np.int32)
    for r, (b0, b1) in enumerate(boxes):
        assert all(0 <= b0[a] < b1[a] <= g[a] for a in range(3))
        sl = owner[b0[2]:b1[2], b0[1]:b1[1], b0[0]:b1[0]]
        assert (sl == -1).all(), "boxes overlap"
        sl[...] = r
    assert (owner >= 0).all(), "bricks left out"

    def leaves(t):
        return [t[1]] if t[0] == "leaf" else leaves(t[3]) + leaves(t[4])

    assert leaves(tree) == list(range(nparts))   # numbered low side first


@pytest.mark.parametrize("impl", IMPLS, ids=lambda i: i.name)
def test_kd_partition_splits_the_longest_axis_into_equal_volumes(impl):
    boxes, tree = impl.kd_partition((64, 128, 256), 16, 2)
    assert tree[1] == 2 and boxes == [((0, 0, 0), (4, 8, 8)), ((0, 0, 8), (4, 8, 16))]
    boxes, _ = impl.kd_partition((64, 128, 256), 16, 8)   # z, then z again (128 = y), then y: 64 x 64 x 64 each
    vol = [np.prod([b1[a] - b0[a] for a in range(3)]) for b0, b1 in boxes]
    assert len(set(vol)) == 1 and all(tuple(b1[a] - b0[a] for a in range(3)) == (4, 4, 4) for b0, b1 in boxes)
    # the paper's cube on 8 GPUs: 512 x 512 x 6400 in 256^3 bricks = 2 x 2 x 25 bricks; parts differ by one slab
    boxes, _ = impl.kd_partition((512, 512, 6400), 256, 8)
    slabs = [b1[2] - b0[2] for b0, b1 in boxes]
    assert sum(slabs) == 25 and max(slabs) - min(slabs) <= 1 and all(b1[0] - b0[0] == 2 and b1[1] - b0[1] == 2 for b0, b1 in boxes)


@pytest.mark.parametrize("impl", IMPLS, ids=lambda i: i.name)
def test_kd_partition_shares_the_longest_axis_between_trees_by_rank_count(impl):
    """6 ranks = a tree of 4 and a tree of 2: the root cut gives the first tree 4/6 of the longest axis."""
    boxes, tree = impl.kd_partition((64, 64, 384), 16, 6)
    assert tree[0] == "node" and tree[1] == 2 and tree[2] == 16     # 24 bricks along z: 16 | 8
    vol = [int(np.prod([b1[a] - b0[a] for a in range(3)])) for b0, b1 in boxes]
    assert vol == [64] * 6                                          # and every rank still holds the same volume
    with pytest.raises(ValueError):
        impl.kd_partition((32, 32, 32), 16, 9)                      # 8 bricks


def test_part_region_adds_the_ghost_layers_inside_the_volume():
    assert sortlast.part_region((64, 64, 64), 16, 2, ((0, 0, 2), (4, 4, 4))) == ((0, 0, 30), (64, 64, 34))
    assert sortlast.part_region((60, 64, 64), 16, 1, ((2, 0, 0), (4, 2, 4))) == ((31, 0, 0), (29, 33, 64))


# --------------------------------------------------------------------------------- visibility order of the parts
def _ray_box(o, d, lo, hi):
    t0, t1 = -np.inf, np.inf
    for a in range(3):
        if d[a] == 0.0:
            if not (lo[a] <= o[a] <= hi[a]):
                return None
            continue
        ta, tb = (lo[a] - o[a]) / d[a], (hi[a] - o[a]) / d[a]
        t0, t1 = max(t0, min(ta, tb)), min(t1, max(ta, tb))
    return (t0, t1) if t1 > max(t0, 0.0) + 1e-9 else None


@pytest.mark.parametrize("impl", IMPLS, ids=lambda i: i.name)
@pytest.mark.parametrize("nparts", [2, 3, 5, 8])
@pytest.mark.parametrize("ortho", [False, True])
def test_part_order_is_a_visibility_order(impl, nparts, ortho):
    """Brute force: along random rays of random cameras (eyes inside the volume included), the parts a ray crosses
    are met in the order part_order lists them."""
    dims, brick = (96, 64, 80), 16
    boxes, tree = impl.kd_partition(dims, brick, nparts)
    rng = np.random.default_rng(7 + nparts)
    fr = synth.Framing(*dims, 64, 48)
    for case in range(40):
        if not ortho and case % 4 == 3:
            eye = tuple(dims[a] * rng.uniform(0.1, 0.9) for a in range(3))
            view, proj = synth.look_at(eye, (0.0, 0.0, 0.0), (0.0, 0.3, 1.0)), synth.perspective(60, 4 / 3, 0.3, 400.0)
        else:
            view, proj = fr.seeded(100 + case, case), fr.proj(ortho)
        order = impl.part_order(tree, brick, view, proj)
        assert sorted(order) == list(range(nparts))
        pos = {r: i for i, r in enumerate(order)}
        Minv = np.linalg.inv(np.asarray(proj, np.float64).reshape(4, 4).T @ np.asarray(view, np.float64).reshape(4, 4).T)
        for _ in range(50):
            x, y = rng.uniform(-1, 1, 2)
            a, b = Minv @ np.array([x, y, -1.0, 1.0]), Minv @ np.array([x, y, 1.0, 1.0])
            o, d = a[:3] / a[3], b[:3] / b[3] - a[:3] / a[3]
            hits = []
            for r, (b0, b1) in enumerate(boxes):
                lo = [b0[k] * brick for k in range(3)]
                hi = [min(b1[k] * brick, dims[k]) for k in range(3)]
                t = _ray_box(o, d, lo, hi)
                if t is not None:
                    hits.append((max(t[0], 0.0), r))
            hits.sort()
            seq = [pos[r] for _, r in hits]
            assert seq == sorted(seq), (case, order, hits)


def test_libvr_partition_and_part_order_equal_the_oracle():
    """vr_kd_partition / vr_part_order against oracle/parts.py: same boxes, same tree, same order, on ragged grids, every
    part count the grid allows up to 12, perspective and orthographic views, eyes inside the volume."""
    rng = np.random.default_rng(11)
    for dims, brick in (((96, 64, 80), 16), ((100, 37, 64), 16), ((33, 200, 90), 8), ((4096, 4096, 1536), 512), ((70, 50, 64), 16)):
        g = sortlast.brick_grid(dims, brick)
        fr = synth.Framing(*dims, 64, 48)
        for nparts in range(1, min(12, g[0] * g[1] * g[2]) + 1):
            try:
                oboxes, otree = oparts.kd_partition(dims, brick, nparts)
            except ValueError:
                with pytest.raises(vr.VrError):
                    sortlast.kd_partition(dims, brick, nparts)
                continue
            boxes, flat = sortlast.kd_partition(dims, brick, nparts)
            assert boxes == oboxes and np.array_equal(flat, oparts.flatten(otree))
            for case in range(8):
                if case % 4 == 3:
                    eye = tuple(dims[a] * rng.uniform(0.05, 0.95) for a in range(3))
                    view, proj = synth.look_at(eye, (0.0, 0.0, 0.0), (0.0, 0.3, 1.0)), synth.perspective(60, 4 / 3, 0.3, 9000.0)
                else:
                    view, proj = fr.seeded(300 + case, case), fr.proj(case % 2 == 1)
                assert sortlast.part_order(flat, brick, view, proj) == oparts.part_order(otree, brick, view, proj)
    with pytest.raises(vr.VrError):
        sortlast.part_order(np.array([[0, 1, 5, 6]], dtype=np.int32), 16, view, proj)   # children outside the tree


# --------------------------------------------------------------------------------- part rectangles (host arithmetic of libvr)
def test_part_rect_contains_the_rendering_rectangles_of_its_bricks():
    dims, brick, W, H = (70, 50, 64), 16, 160, 120
    o = oracle.Volume(*dims, brick, 1, data=np.zeros(dims[::-1], dtype=np.float32))
    g = sortlast.brick_grid(dims, brick)
    fr = synth.Framing(*dims, W, H)
    for nparts in (2, 3, 4):
        boxes, _ = sortlast.kd_partition(dims, brick, nparts)
        for case in range(6):
            view, proj = fr.seeded(40 + case, case), fr.proj(case % 2 == 1)
            rects = o.rects(view, proj, W, H)
            for b0, b1 in boxes:
                pr = vr.part_rect(dims, brick, (b0, b1), view, proj, W, H)
                own = [rects[(bz * g[1] + by) * g[0] + bx] for bz in range(b0[2], b1[2]) for by in range(b0[1], b1[1])
                       for bx in range(b0[0], b1[0])]
                own = np.array([r for r in own if r[2] > r[0] and r[3] > r[1]])
                u = (own[:, 0].min(), own[:, 1].min(), own[:, 2].max(), own[:, 3].max())
                assert pr[0] <= u[0] and pr[1] <= u[1] and pr[2] >= u[2] and pr[3] >= u[3]       # contains
                assert pr[0] >= u[0] - 1 and pr[1] >= u[1] - 1 and pr[2] <= u[2] + 1 and pr[3] <= u[3] + 1  # one pixel of slack
    with pytest.raises(vr.VrError):
        vr.part_rect(dims, brick, ((0, 0, 0), (9, 1, 1)), view, proj, W, H)


# --------------------------------------------------------------------------------- the protocol over gloo
class OracleBackend:
    """Test stand-in for the two kernels around the exchange: the pieces of a partial frame from the oracle's per-brick
    sub-images (ALPHA: premultiplied RGBA; MIP: ONE float per pixel, the raw maximum, -inf without a sample -
    PAPER.md:180), merging with the oracle's compositor (MIP: maximum, then the colour mapping)."""

    def __init__(self, vol, dims, brick, box, tf):
        self.vol, self.dims, self.brick, self.box, self.tf = vol, dims, brick, box, np.asarray(tf, dtype=np.float64)
        self.device = torch.device("cpu")
        g = sortlast.brick_grid(dims, brick)
        self.own = [(bz * g[1] + by) * g[0] + bx for bz in range(box[0][2], box[1][2]) for by in range(box[0][1], box[1][1])
                    for bx in range(box[0][0], box[1][0])]

    def empty(self, shape):
        return torch.empty(shape, dtype=torch.float32)

    def empty_piece(self, rect, mode):
        h, w = rect[3] - rect[1], rect[2] - rect[0]
        return self.empty((h, w, 4) if mode == oracle.ALPHA else (h, w))

    def render_pieces(self, view, proj, W, H, step, mode, rects):
        ref = self.vol.render(view, proj, W, H, step, mode, want_sub=True)
        sub = ref["sub"].reshape(H, W, -1, 4)
        order = [b for b in self.vol.brick_order(view, proj) if b in set(self.own)]
        if mode == oracle.ALPHA:
            acc = np.zeros((H, W, 4))
            for b in order:
                acc += (1.0 - acc[..., 3:4]) * sub[:, :, b]
        else:
            acc = sub[:, :, self.own, 0].max(axis=2)
        # nothing of the part lies outside its rectangle: the pieces lose nothing
        pr = vr.part_rect(self.dims, self.brick, self.box, view, proj, W, H)
        outside = np.ones((H, W), dtype=bool)
        outside[pr[1]:pr[3], pr[0]:pr[2]] = False
        assert not (np.isfinite(acc) & (acc != 0)).reshape(H, W, -1).any(axis=-1)[outside].any()
        return [torch.from_numpy(np.ascontiguousarray(acc[r[1]:r[3], r[0]:r[2]], dtype=np.float32)) for r in rects]

    def composite_parts(self, mode, pieces, rects, order, W, H):
        if mode == oracle.ALPHA:
            out = oracle.composite([p.numpy() for p in pieces], rects, order, W, H)
        else:
            m = np.full((H, W), -np.inf)
            for p, r in zip(pieces, rects):
                sl = m[r[1]:r[3], r[0]:r[2]]
                sl[...] = np.maximum(sl, p.numpy().astype(np.float64))
            n = self.tf.shape[0]
            x = np.clip((m - synth.TF_VMIN) / (synth.TF_VMAX - synth.TF_VMIN), 0.0, 1.0) * (n - 1)
            x = np.where(np.isfinite(m), x, 0.0)
            i = np.minimum(np.floor(x).astype(np.int64), n - 2)
            f = (x - i)[..., None]
            out = self.tf[i] + f * (self.tf[i + 1] - self.tf[i])
            out[..., 3] = 1.0
            out[~np.isfinite(m)] = 0.0
        return torch.from_numpy(np.ascontiguousarray(out, dtype=np.float32))


DIMS, BRICK, W, H = (40, 33, 48), 16, 72, 54


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group(backend="gloo", rank=rank, world_size=world)
    cube = synth.Cube(11, *DIMS, 3)
    vol = oracle.Volume(*DIMS, BRICK, 1, data=cube.fill_host())
    vol.set_transfer_function(synth.tf_translucent(), synth.TF_VMIN, synth.TF_VMAX)
    vol.set_early_termination(2.0)
    boxes, _ = sortlast.kd_partition(DIMS, BRICK, world)
    rdr = sortlast.SortLastRenderer(DIMS, BRICK, 1, backend=OracleBackend(vol, DIMS, BRICK, boxes[rank], synth.tf_translucent()))
    fr = synth.Framing(*DIMS, W, H)
    worst = []
    for case in range(4):
        view, proj = fr.seeded(60 + case, case), fr.proj(case == 3)
        for mode in (oracle.ALPHA, oracle.MIP):
            frame = rdr.render(view, proj, W, H, 0.7, mode)
            if rank == 0:
                ref = vol.render(view, proj, W, H, 0.7, mode)
                worst.append(float(np.abs(frame.numpy() - ref["image"]).max()))  # MIP: the colour-mapped frame (R11)
            else:
                assert frame is None
    moved = rdr.exchange_bytes(view, proj, W, H, oracle.ALPHA)
    moved_mip = rdr.exchange_bytes(view, proj, W, H, oracle.MIP)
    stripes_to_rank0 = sum((y1 - y0) * W * 16 for (y0, y1) in sortlast.stripes(H, world)[1:])
    assert (moved_mip - stripes_to_rank0) * 4 == moved - stripes_to_rank0   # MIP pieces travel as one float per pixel
    out.put((rank, worst, moved))
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.parametrize("world", [2, 3])
def test_exchange_protocol_over_gloo(world):
    port = _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=300) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    worst = res[0][1]
    assert len(worst) == 8 and max(worst) < 2e-6, worst      # float32 partial frames against the double-precision frame
    M = W * H * 16
    assert all(r[2] == res[0][2] for r in res) and res[0][2] < 2 * M   # "M + epsilon", not N x M


def test_a_world_of_one_needs_no_process_group():
    cube = synth.Cube(11, *DIMS, 3)
    vol = oracle.Volume(*DIMS, BRICK, 1, data=cube.fill_host())
    vol.set_transfer_function(synth.tf_ramp(), synth.TF_VMIN, synth.TF_VMAX)
    boxes, _ = sortlast.kd_partition(DIMS, BRICK, 1)
    rdr = sortlast.SortLastRenderer(DIMS, BRICK, 1, backend=OracleBackend(vol, DIMS, BRICK, boxes[0], synth.tf_ramp()), rank=0, world=1)
    fr = synth.Framing(*DIMS, W, H)
    view, proj = fr.seeded(5, 0), fr.proj(False)
    frame = rdr.render(view, proj, W, H, 1.0, oracle.ALPHA)
    assert np.abs(frame.numpy() - vol.render(view, proj, W, H, 1.0, oracle.ALPHA)["image"]).max() < 2e-6


def test_the_product_backend_refuses_to_run_without_a_gpu():
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    with pytest.raises(RuntimeError):
        sortlast.SortLastRenderer(DIMS, BRICK, 1, rank=0, world=1)
