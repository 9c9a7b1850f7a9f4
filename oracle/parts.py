"""oracle.parts -- TEST INFRASTRUCTURE: plain statement of the data partition and part visibility order of the
multi-GPU sort-last renderer, the counterpart of libvr's vr_kd_partition / vr_part_order.

PAPER.md:138 (sec. 2.3.1): the cube is dealt to the GPUs with k-d trees (balanced binary splits; several trees when
the GPU count is not a power of two). PAPER.md:174: alpha blending is associative, so partial frames composite in
visibility order. Readings (the paper gives no rule for the cuts): a box of bricks is cut across its longest axis
(in voxels, ties to the lower axis) at the brick face nearest to the wanted share (round half to even), at least one
brick per side; n = 2^k parts make one balanced tree, other counts a chain of balanced trees, one per set bit of n
from the largest down, whose roots share the box in proportion to their leaf counts. Visibility: at every node the
side of the cut plane that holds the eye comes first (orthographic: the side the view direction leaves first); the
eye is R9's homogeneous eye, here from numpy's own inverse.

Pinned by tests/test_sortlast.py: the boxes tile the brick grid; the paper-rule cases (longest axis first, equal
halves, 6 = 4 + 2); the order is a visibility order by brute force along random rays, eyes inside the volume included.
Shares no code with paper_1205_0282_b200 (which does this in C++, csrc/vr_parts.cu).
"""
import numpy as np


def brick_grid(dims, brick):
    return tuple((int(n) + int(brick) - 1) // int(brick) for n in dims)


def _extent(dims, brick, lo, hi, a):
    """Voxels of bricks [lo, hi) along axis a (the last brick of an axis may be ragged)."""
    return min(hi * brick, dims[a]) - lo * brick


def _split(dims, brick, b0, b1, n_low, n_all):
    axes = sorted(range(3), key=lambda a: (-_extent(dims, brick, b0[a], b1[a], a), a))
    for a in axes:
        if b1[a] - b0[a] < 2:
            continue
        want = b0[a] * brick + _extent(dims, brick, b0[a], b1[a], a) * n_low / n_all
        cut = int(round(want / brick))
        return a, min(max(cut, b0[a] + 1), b1[a] - 1)
    raise ValueError("more parts than bricks in the box %s..%s" % (b0, b1))


def _balanced(dims, brick, b0, b1, n, first, boxes):
    if n == 1:
        boxes[first] = (tuple(b0), tuple(b1))
        return ("leaf", first)
    a, cut = _split(dims, brick, b0, b1, 1, 2)
    lo1, hi0 = list(b0), list(b1)
    hi0[a] = cut
    lo1[a] = cut
    return ("node", a, cut, _balanced(dims, brick, b0, hi0, n // 2, first, boxes),
            _balanced(dims, brick, lo1, b1, n // 2, first + n // 2, boxes))


def kd_partition(dims, brick, nparts):
    """Returns (boxes, tree): boxes[r] = (b0, b1), the half-open brick box of part r; tree = nested
    ("node", axis, cut, low, high) / ("leaf", r) with the cut in brick units."""
    nparts = int(nparts)
    if nparts < 1:
        raise ValueError("nparts must be positive")
    g = brick_grid(dims, brick)
    if nparts > g[0] * g[1] * g[2]:
        raise ValueError("%d parts for %d bricks" % (nparts, g[0] * g[1] * g[2]))
    boxes = [None] * nparts
    sizes = [1 << k for k in range(nparts.bit_length() - 1, -1, -1) if nparts >> k & 1]  # 6 -> [4, 2]

    def forest(b0, b1, sizes, first):
        if len(sizes) == 1:
            return _balanced(dims, brick, b0, b1, sizes[0], first, boxes)
        a, cut = _split(dims, brick, b0, b1, sizes[0], sum(sizes))
        lo1, hi0 = list(b0), list(b1)
        hi0[a] = cut
        lo1[a] = cut
        return ("node", a, cut, _balanced(dims, brick, b0, hi0, sizes[0], first, boxes),
                forest(lo1, b1, sizes[1:], first + sizes[0]))

    tree = forest([0, 0, 0], list(g), sizes, 0)
    return boxes, tree


def eye_of(view, proj):
    """R9's homogeneous eye: third column of (proj*view)^-1. Returns (xyz, ortho)."""
    V = np.asarray(view, dtype=np.float32).astype(np.float64).reshape(4, 4).T  # column-major input
    P = np.asarray(proj, dtype=np.float32).astype(np.float64).reshape(4, 4).T
    c = np.linalg.inv(P @ V)[:, 2]
    if abs(c[3]) < 1e-9 * np.abs(c[:3]).sum():
        return c[:3], True
    return c[:3] / c[3], False


def part_order(tree, brick, view, proj):
    """The parts front to back: at every node the side that holds the eye first."""
    eye, ortho = eye_of(view, proj)
    out = []

    def walk(t):
        if t[0] == "leaf":
            out.append(t[1])
            return
        _, a, cut, low, high = t
        low_first = eye[a] >= 0.0 if ortho else eye[a] < cut * brick
        walk(low if low_first else high)
        walk(high if low_first else low)

    walk(tree)
    return out


def flatten(tree):
    """The nested tree in libvr's encoding (pre-order rows (axis, cut, low, high) / (-1, part, 0, 0)), for comparison."""
    rows = []

    def walk(t):
        me = len(rows)
        rows.append(None)
        if t[0] == "leaf":
            rows[me] = (-1, t[1], 0, 0)
        else:
            lo = walk(t[3])
            hi = walk(t[4])
            rows[me] = (t[1], t[2], lo, hi)
        return me

    walk(tree)
    return np.array(rows, dtype=np.int32)
