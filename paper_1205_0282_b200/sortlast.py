"""Multi-GPU sort-last rendering: one process per GPU, each holding a box of bricks.

The paper's scheme (PAPER.md:136-138 partitioning, :170-174 two-stage compositing, :178-184 direct send of
rectangle-packed partial frames), mapped onto one node of B200s:

  1. `vr_kd_partition` deals the brick grid to the ranks as boxes: balanced k-d trees, split across the longest
     axis, and for a rank count that is not a power of two several trees whose roots share the longest axis in
     proportion to their rank counts.
  2. The frame is dealt to the ranks in horizontal stripes; rank r owes rank s the piece rect(r) ∩ stripe(s) of its
     partial frame, where rect(r) is the part's rendering rectangle (`vr_part_rect`, computed by every rank for every
     part from the geometry alone: no size handshake). Every rank renders its own bricks and composites them
     straight INTO those rectangle-packed pieces (`vr_render_part_pieces`: stage-1 compositing on the GPU that
     rendered, "each node utilizes its local memory to do the first local composition") - float4 per pixel
     for ALPHA, ONE float per pixel for MIP as in the paper (:180: 4 MB per 1024^2 sub-frame).
  3. The pieces travel: the volume moved per frame is the frame size plus the overlap of the rectangles,
     "M + epsilon". This is a direct send: point-to-point `torch.distributed`
     messages, NCCL over NVLink on GPUs.
  4. Every rank merges the pieces of its stripe in part visibility order (`vr_composite_parts`: `over` for
     ALPHA, which NCCL's reductions cannot express; maximum + colour mapping for MIP) and rank 0 collects the
     stripes.

This module is plumbing: the arithmetic of every step runs in libvr's kernels through the `backend` (default: a
part handle on the current CUDA device). Tests pass a backend of their own to run the protocol over gloo on CPUs.
"""
from . import ALPHA, MIP, Volume, kd_partition, part_order, part_rect  # noqa: F401 (kd_partition, part_order: re-exported)


# ---------------------------------------------------------------------------------------------------------------
# which voxels a rank uploads, which rows it merges (index bookkeeping; the partition and the part order are libvr's
# vr_kd_partition / vr_part_order, the rectangles vr_part_rect)
# ---------------------------------------------------------------------------------------------------------------
def brick_grid(dims, brick):
    return tuple((int(n) + int(brick) - 1) // int(brick) for n in dims)


def part_region(dims, brick, ghost, box):
    """The voxels a part needs uploaded: its bricks plus `ghost` layers of its neighbours', clipped to the volume.
    Returns (origin, shape) in (x, y, z) order."""
    lo = [max(box[0][a] * brick - ghost, 0) for a in range(3)]
    hi = [min(min(box[1][a] * brick, dims[a]) + ghost, dims[a]) for a in range(3)]
    return tuple(lo), tuple(h - l for l, h in zip(lo, hi))


def stripes(height, nparts):
    """Rows [y0, y1) of the frame each rank merges."""
    return [(height * r // nparts, height * (r + 1) // nparts) for r in range(nparts)]


def _clip(rect, y0, y1):
    r = (rect[0], max(rect[1], y0), rect[2], min(rect[3], y1))
    return r if r[2] > r[0] and r[3] > r[1] else None


# ---------------------------------------------------------------------------------------------------------------
# the renderer
# ---------------------------------------------------------------------------------------------------------------
class CudaBackend:
    """The product backend: a part handle of libvr on the current CUDA device."""

    def __init__(self, dims, brick, ghost, box):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("paper_1205_0282_b200.sortlast needs a CUDA device (libvr has no CPU path)")
        self.torch = torch
        self.device = torch.device("cuda", torch.cuda.current_device())
        self.volume = Volume(dims[0], dims[1], dims[2], brick, ghost, part=box)

    def empty(self, shape):
        return self.torch.empty(shape, dtype=self.torch.float32, device=self.device)

    def empty_piece(self, rect, mode):
        h, w = rect[3] - rect[1], rect[2] - rect[0]
        return self.empty((h, w, 4) if mode == ALPHA else (h, w))

    def render_pieces(self, view, proj, width, height, step, mode, rects):
        """The part's partial frame as one tensor per rectangle: [h][w][4] (ALPHA) or [h][w] (MIP, raw maximum)."""
        pieces = [self.empty_piece(r, mode) for r in rects]
        self.volume.render_part_pieces(view, proj, width, height, step, mode, rects, pieces)
        return pieces

    def composite_parts(self, mode, pieces, rects, order, width, height):
        out = self.empty((height, width, 4))
        return self.volume.composite_parts(mode, pieces, rects, order, width, height, out)


class SortLastRenderer:
    """One rank of a sort-last renderer. `group`: a torch.distributed process group (None = the default one; a
    world of one works without torch.distributed). Collective: every rank calls every method."""

    def __init__(self, dims, brick, ghost=1, group=None, backend=None, rank=None, world=None):
        self.dims, self.brick, self.ghost, self.group = tuple(int(n) for n in dims), int(brick), int(ghost), group
        if rank is None:
            import torch.distributed as dist
            if dist.is_available() and dist.is_initialized():
                rank, world = dist.get_rank(group), dist.get_world_size(group)
            else:
                rank, world = 0, 1
        self.rank, self.world = int(rank), int(world)
        self.boxes, self.tree = kd_partition(self.dims, self.brick, self.world)
        self.box = self.boxes[self.rank]
        self.backend = backend if backend is not None else CudaBackend(self.dims, self.brick, self.ghost, self.box)

    # -- data --------------------------------------------------------------------------------------------------
    def region(self):
        """(origin, shape), x-y-z: the voxels this rank has to upload (its bricks and their ghost layers)."""
        return part_region(self.dims, self.brick, self.ghost, self.box)

    def upload(self, data, origin):
        """data: float32 [sz][sy][sx] of the region (or any box of the volume: what the part does not hold is ignored)."""
        self.backend.volume.upload(data, origin=origin)

    def set_transfer_function(self, rgba, vmin, vmax):
        self.backend.volume.set_transfer_function(rgba, vmin, vmax)

    def set_early_termination(self, tau):
        self.backend.volume.set_early_termination(tau)

    def minmax(self):
        """The data range of the whole volume: the parts' ranges, reduced over the ranks."""
        lo, hi = self.backend.volume.minmax()
        if self.world > 1:
            import torch
            import torch.distributed as dist
            t = torch.tensor([-lo, hi], dtype=torch.float32, device=self.backend.device)
            dist.all_reduce(t, op=dist.ReduceOp.MAX, group=self.group)
            lo, hi = -float(t[0]), float(t[1])
        return lo, hi

    # -- one frame -----------------------------------------------------------------------------------------------
    def render(self, view, proj, width, height, step, mode):
        """Returns the frame [height][width][4] on rank 0 (a tensor on the backend's device), None elsewhere."""
        if mode not in (ALPHA, MIP):
            raise ValueError("SortLastRenderer.render: mode must be ALPHA or MIP")
        be, R, me = self.backend, self.world, self.rank
        rects = [part_rect(self.dims, self.brick, b, view, proj, width, height) for b in self.boxes]
        order = part_order(self.tree, self.brick, view, proj)
        rows = stripes(height, R)

        def piece_of(r, s):
            return _clip(rects[r], rows[s][0], rows[s][1])

        # stage 1 on this GPU, straight into the pieces this rank owes every stripe (its own included)
        owed = [(s, piece_of(me, s)) for s in range(R)]
        owed = [(s, c) for s, c in owed if c is not None]
        rendered = be.render_pieces(view, proj, width, height, step, mode, [c for _, c in owed])
        mine = dict((s, t) for (s, _), t in zip(owed, rendered))
        pieces = {}  # source rank -> tensor of rect(r) ∩ my stripe
        if me in mine:
            pieces[me] = mine[me]
        if R > 1:
            import torch.distributed as dist
            ops = []
            for s in range(R):
                if s == me:
                    continue
                if s in mine:  # direct send of the packed piece
                    ops.append(dist.P2POp(dist.isend, mine[s], self._global(s), group=self.group))
                c = piece_of(s, me)
                if c is not None:
                    pieces[s] = be.empty_piece(c, mode)
                    ops.append(dist.P2POp(dist.irecv, pieces[s], self._global(s), group=self.group))
            if ops:
                for w in dist.batch_isend_irecv(ops):
                    w.wait()
        # merge my stripe, front to back; rectangles in stripe coordinates
        y0, y1 = rows[me]
        src = [r for r in order if r in pieces]
        local = []
        for r in src:
            c = piece_of(r, me)
            local.append((c[0], c[1] - y0, c[2], c[3] - y0))
        stripe = None
        if y1 > y0:
            stripe = be.composite_parts(mode, [pieces[r] for r in src], local, list(range(len(src))), width, y1 - y0)
        if R == 1:
            return stripe
        # collect the stripes on rank 0
        import torch.distributed as dist
        if me == 0:
            frame = be.empty((height, width, 4))
            if stripe is not None:
                frame[y0:y1] = stripe
            ops = [dist.P2POp(dist.irecv, frame[rows[s][0]:rows[s][1]], self._global(s), group=self.group)
                   for s in range(1, R) if rows[s][1] > rows[s][0]]
            if ops:
                for w in dist.batch_isend_irecv(ops):
                    w.wait()
            return frame
        if stripe is not None:
            for w in dist.batch_isend_irecv([dist.P2POp(dist.isend, stripe, self._global(0), group=self.group)]):
                w.wait()
        return None

    def _global(self, r):
        if self.group is None:
            return r
        import torch.distributed as dist
        return dist.get_global_rank(self.group, r)

    def exchange_bytes(self, view, proj, width, height, mode=ALPHA):
        """Bytes this frame's exchange moves between ranks (pieces sent to other ranks: 16 bytes per pixel for ALPHA, 4 for
        MIP; + the merged RGBA stripes sent to rank 0): the paper's M + epsilon, from the geometry alone."""
        rects = [part_rect(self.dims, self.brick, b, view, proj, width, height) for b in self.boxes]
        rows = stripes(height, self.world)
        total = 0
        for r in range(self.world):
            for s in range(self.world):
                c = _clip(rects[r], rows[s][0], rows[s][1])
                if r != s and c is not None:
                    total += (c[2] - c[0]) * (c[3] - c[1]) * (16 if mode == ALPHA else 4)
        total += sum((y1 - y0) * width * 16 for (y0, y1) in rows[1:])
        return total
