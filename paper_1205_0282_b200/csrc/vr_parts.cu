/*
 * vr_parts.cu -- data partitioning and part visibility order of the multi-GPU sort-last renderer
 * (SURVEY.md sec. 8(e), row f3). Host arithmetic: every process computes the same partition and the
 * same order from the geometry alone, no message is needed.
 *
 * PAPER.md:138 (sec. 2.3.1): the cube is dealt to the GPUs with k-d trees - balanced binary splits,
 * and for a GPU count that is not a power of two several trees. Here: the brick grid is cut across
 * its longest axis (in voxels; ties to the lower axis) at a brick face until every part is a box of
 * bricks; nparts = 2^k gives one balanced tree, any other count a chain of balanced trees, one per
 * set bit of nparts from the largest down, whose roots share the box in proportion to their leaf
 * counts (6 = 4 + 2: the first cut puts 4/6 of the longest axis on the low side).
 * `over` needs the partial frames front to back. The boxes on the two sides of a cut
 * are separated by the cut plane, so visiting the side that holds the eye first - at every node -
 * is a visibility order of the parts (orthographic: the side the view direction leaves first); the
 * eye is R9's homogeneous eye from the library's own Gauss-Jordan inverse (vr_view.cuh).
 *
 * Tree encoding (host int[(2 * nparts - 1) * 4], node 0 = root, pre-order): an inner node is
 * (axis, cut, low child, high child) with the cut in BRICK units; a leaf is (-1, part, 0, 0).
 */
#include <math.h>
#include <string.h>

#include "vr_view.cuh"

struct PartBuild {
    int n[3], brick;
    int* boxes; /* nparts * 6 */
    int* tree;  /* (2 nparts - 1) * 4 */
    int next_node;
};

static int extent_of(const PartBuild& B, int lo, int hi, int a) {
    const long long top = (long long)hi * B.brick;
    return (int)((top < B.n[a] ? top : B.n[a]) - (long long)lo * B.brick);
}

/* cut of the box across its longest axis with more than one brick; the low side gets n_low / n_all of the extent,
 * rounded to a brick face (ties to even, as rint does), at least one brick on each side. Returns the axis or -1. */
static int split_of(const PartBuild& B, const int b0[3], const int b1[3], int n_low, int n_all, int* cut) {
    int axes[3] = {0, 1, 2};
    for (int i = 0; i < 3; ++i)
        for (int j = i + 1; j < 3; ++j) {
            const int ei = extent_of(B, b0[axes[i]], b1[axes[i]], axes[i]), ej = extent_of(B, b0[axes[j]], b1[axes[j]], axes[j]);
            if (ej > ei || (ej == ei && axes[j] < axes[i])) {
                const int t = axes[i];
                axes[i] = axes[j];
                axes[j] = t;
            }
        }
    for (int i = 0; i < 3; ++i) {
        const int a = axes[i];
        if (b1[a] - b0[a] < 2) continue;
        const double want = (double)((long long)b0[a] * B.brick) + (double)((long long)extent_of(B, b0[a], b1[a], a) * n_low) / (double)n_all;
        int c = (int)rint(want / (double)B.brick);
        if (c < b0[a] + 1) c = b0[a] + 1;
        if (c > b1[a] - 1) c = b1[a] - 1;
        *cut = c;
        return a;
    }
    return -1;
}

/* balanced tree with n = 2^k leaves numbered first, first + 1, ... low side first; returns its node or -1 */
static int balanced(PartBuild& B, const int b0[3], const int b1[3], int n, int first) {
    const int me = B.next_node++;
    int* t = B.tree + 4 * me;
    if (n == 1) {
        for (int a = 0; a < 3; ++a) B.boxes[6 * first + a] = b0[a], B.boxes[6 * first + 3 + a] = b1[a];
        t[0] = -1; t[1] = first; t[2] = 0; t[3] = 0;
        return me;
    }
    int cut = 0;
    const int a = split_of(B, b0, b1, 1, 2, &cut);
    if (a < 0) return -1;
    int hi0[3] = {b1[0], b1[1], b1[2]}, lo1[3] = {b0[0], b0[1], b0[2]};
    hi0[a] = cut;
    lo1[a] = cut;
    const int lo = balanced(B, b0, hi0, n / 2, first);
    const int hi = lo < 0 ? -1 : balanced(B, lo1, b1, n / 2, first + n / 2);
    if (lo < 0 || hi < 0) return -1;
    t[0] = a; t[1] = cut; t[2] = lo; t[3] = hi;
    return me;
}

static int forest(PartBuild& B, const int b0[3], const int b1[3], const int* sizes, int nsizes, int first) {
    if (nsizes == 1) return balanced(B, b0, b1, sizes[0], first);
    int all = 0;
    for (int i = 0; i < nsizes; ++i) all += sizes[i];
    const int me = B.next_node++;
    int cut = 0;
    const int a = split_of(B, b0, b1, sizes[0], all, &cut);
    if (a < 0) return -1;
    int hi0[3] = {b1[0], b1[1], b1[2]}, lo1[3] = {b0[0], b0[1], b0[2]};
    hi0[a] = cut;
    lo1[a] = cut;
    const int lo = balanced(B, b0, hi0, sizes[0], first);
    const int hi = lo < 0 ? -1 : forest(B, lo1, b1, sizes + 1, nsizes - 1, first + sizes[0]);
    if (lo < 0 || hi < 0) return -1;
    int* t = B.tree + 4 * me;
    t[0] = a; t[1] = cut; t[2] = lo; t[3] = hi;
    return me;
}

int vr_host_kd_partition(int nx, int ny, int nz, int brick, int nparts, int* boxes_out, int* tree_out) {
    PartBuild B;
    B.n[0] = nx; B.n[1] = ny; B.n[2] = nz;
    B.brick = brick;
    B.boxes = boxes_out;
    B.tree = tree_out;
    B.next_node = 0;
    int g[3], zero[3] = {0, 0, 0};
    for (int a = 0; a < 3; ++a) g[a] = (B.n[a] + brick - 1) / brick;
    int sizes[32], ns = 0;
    for (int k = 30; k >= 0; --k)
        if (nparts >> k & 1) sizes[ns++] = 1 << k;
    return forest(B, zero, g, sizes, ns, 0) == 0 ? 0 : 1;
}

int vr_host_part_order(const int* tree, int nparts, int brick, const float* view, const float* proj, int* order_out) {
    double M[16], Minv[16], eye[3];
    int ortho = 0;
    if (vr_view_setup(view, proj, M, Minv, eye, &ortho)) return 1;
    const int nnodes = 2 * nparts - 1;
    int stack[64], sp = 0, n = 0;
    stack[sp++] = 0;
    while (sp > 0) {
        const int t = stack[--sp];
        if (t < 0 || t >= nnodes) return 2;
        const int* nd = tree + 4 * t;
        if (nd[0] < 0) {
            if (nd[1] < 0 || nd[1] >= nparts || n >= nparts) return 2;
            order_out[n++] = nd[1];
            continue;
        }
        if (nd[0] > 2 || sp + 2 > 64) return 2;
        const bool low_first = ortho ? eye[nd[0]] >= 0.0 : eye[nd[0]] < (double)nd[1] * (double)brick;
        stack[sp++] = low_first ? nd[3] : nd[2]; /* popped second: the far side */
        stack[sp++] = low_first ? nd[2] : nd[3];
    }
    return n == nparts ? 0 : 2;
}
