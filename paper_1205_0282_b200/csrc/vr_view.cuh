/*
 * vr_view.cuh -- per-view geometry in IEEE double precision, one rounding per operation.
 *
 * DESIGN.md "Set-up arithmetic" fixes the order of operations of the view set-up (matrix
 * product, Gauss-Jordan inverse, homogeneous eye, rectangle projection, pixel ray, slab
 * test) so that "brick order and ray-brick lists must match exactly" is well posed (R9,
 * R10): every step below is an individually rounded +, -, *, /, sqrt or fma, never a
 * contracted multiply-add. On the device that is enforced with the _rn intrinsics; the host
 * copy (argument validation and scratch sizing only) is compiled with -ffp-contract=off.
 *
 * Paper: PAPER.md:150 (sec. 2.3.2: the viewer's OpenGL projection and transformation
 * matrices; each sub-cube's vertices are projected and their bounding rectangle limits the
 * ray casting), :152 (ray start, orientation, intersection with the bounding cube).
 */
#ifndef VR_VIEW_CUH
#define VR_VIEW_CUH

#include <math.h>

#include "vr_internal.cuh"

#ifdef __CUDA_ARCH__
#define VR_ADD(a, b) __dadd_rn((a), (b))
#define VR_SUB(a, b) __dsub_rn((a), (b))
#define VR_MUL(a, b) __dmul_rn((a), (b))
#define VR_DIV(a, b) __ddiv_rn((a), (b))
#define VR_SQRT(a) __dsqrt_rn((a))
#define VR_FMA(a, b, c) __fma_rn((a), (b), (c))
#else
#define VR_ADD(a, b) ((double)(a) + (double)(b))
#define VR_SUB(a, b) ((double)(a) - (double)(b))
#define VR_MUL(a, b) ((double)(a) * (double)(b))
#define VR_DIV(a, b) ((double)(a) / (double)(b))
#define VR_SQRT(a) sqrt((double)(a))
#define VR_FMA(a, b, c) fma((double)(a), (double)(b), (double)(c))
#endif

#define VR_HD __host__ __device__ __forceinline__

/* C = A * B, column-major 4x4; each entry is ((((0 + t0) + t1) + t2) + t3). */
__host__ __device__ inline void vr_mat_mul(const double* A, const double* B, double* C) {
    for (int c = 0; c < 4; ++c)
        for (int r = 0; r < 4; ++r) {
            double s = 0.0;
            for (int k = 0; k < 4; ++k) s = VR_ADD(s, VR_MUL(A[k * 4 + r], B[c * 4 + k]));
            C[c * 4 + r] = s;
        }
}

/* Gauss-Jordan elimination with partial pivoting on [A | I]; returns 1 if a pivot is 0. */
__host__ __device__ inline int vr_mat_inv(const double* A, double* Ainv) {
    double a[4][8];
    for (int r = 0; r < 4; ++r)
        for (int c = 0; c < 4; ++c) {
            a[r][c] = A[c * 4 + r];
            a[r][4 + c] = (r == c) ? 1.0 : 0.0;
        }
    for (int col = 0; col < 4; ++col) {
        int piv = col;
        for (int r = col + 1; r < 4; ++r)
            if (fabs(a[r][col]) > fabs(a[piv][col])) piv = r;
        if (a[piv][col] == 0.0) return 1;
        if (piv != col)
            for (int c = 0; c < 8; ++c) {
                double t = a[piv][c];
                a[piv][c] = a[col][c];
                a[col][c] = t;
            }
        const double d = a[col][col];
        for (int c = 0; c < 8; ++c) a[col][c] = VR_DIV(a[col][c], d);
        for (int r = 0; r < 4; ++r) {
            if (r == col) continue;
            const double f = a[r][col];
            if (f != 0.0)
                for (int c = 0; c < 8; ++c) a[r][c] = VR_SUB(a[r][c], VR_MUL(f, a[col][c]));
        }
    }
    for (int r = 0; r < 4; ++r)
        for (int c = 0; c < 4; ++c) Ainv[c * 4 + r] = a[r][4 + c];
    return 0;
}

/* M = P*V, Minv, and the homogeneous eye Minv*(0,0,1,0) = third column of Minv (R9):
 * w ~ 0 -> orthographic, xyz is the forward direction; else the eye point xyz/w. */
__host__ __device__ inline int vr_view_setup(const float* view, const float* proj, double* M, double* Minv, double* eye,
                                             int* ortho) {
    double V[16], P[16];
    for (int i = 0; i < 16; ++i) {
        V[i] = (double)view[i];
        P[i] = (double)proj[i];
    }
    vr_mat_mul(P, V, M);
    if (vr_mat_inv(M, Minv)) return 1;
    for (int i = 0; i < 16; ++i)
        if (!isfinite(Minv[i])) return 1;
    const double c0 = Minv[8], c1 = Minv[9], c2 = Minv[10], c3 = Minv[11];
    const double mag = VR_ADD(VR_ADD(fabs(c0), fabs(c1)), fabs(c2));
    if (fabs(c3) < VR_MUL(1e-9, mag)) {
        *ortho = 1;
        eye[0] = c0; eye[1] = c1; eye[2] = c2;
    } else {
        *ortho = 0;
        eye[0] = VR_DIV(c0, c3); eye[1] = VR_DIV(c1, c3); eye[2] = VR_DIV(c2, c3);
    }
    return 0;
}

VR_HD void vr_brick_coords(const VrGrid& g, int b, int bc[3]) {
    bc[0] = b % g.g[0];
    bc[1] = (b / g.g[0]) % g.g[1];
    bc[2] = b / (g.g[0] * g.g[1]);
}

VR_HD void vr_brick_core(const VrGrid& g, const int bc[3], int lo[3], int hi[3]) {
    for (int a = 0; a < 3; ++a) {
        lo[a] = bc[a] * g.brick;
        hi[a] = lo[a] + g.brick;
        if (hi[a] > g.n[a]) hi[a] = g.n[a];
    }
}

/* Rendering rectangle of a box (Fig. 4): bounding rectangle of the 8 projected
 * vertices, half-open pixel ranges clipped to the viewport; a vertex with clip w <= 1e-12
 * makes it the whole viewport. */
__host__ __device__ inline void vr_rect_of_box(const double* M, const int lo[3], const int hi[3], int W, int H, int r[4]) {
    double xmin = INFINITY, xmax = -INFINITY, ymin = INFINITY, ymax = -INFINITY;
    bool full = false;
    for (int c = 0; c < 8; ++c) {
        const double wx = (c & 1) ? (double)hi[0] : (double)lo[0];
        const double wy = (c & 2) ? (double)hi[1] : (double)lo[1];
        const double wz = (c & 4) ? (double)hi[2] : (double)lo[2];
        double q[4];
        for (int k = 0; k < 4; ++k)
            q[k] = VR_ADD(VR_ADD(VR_ADD(VR_MUL(M[k], wx), VR_MUL(M[4 + k], wy)), VR_MUL(M[8 + k], wz)), VR_MUL(M[12 + k], 1.0));
        if (!(q[3] > 1e-12)) {
            full = true;
            break;
        }
        const double px = VR_MUL(VR_MUL(VR_ADD(VR_DIV(q[0], q[3]), 1.0), 0.5), (double)W);
        const double py = VR_MUL(VR_MUL(VR_ADD(VR_DIV(q[1], q[3]), 1.0), 0.5), (double)H);
        if (px < xmin) xmin = px;
        if (px > xmax) xmax = px;
        if (py < ymin) ymin = py;
        if (py > ymax) ymax = py;
    }
    r[0] = 0; r[1] = 0; r[2] = W; r[3] = H;
    if (!full) {
        const double fx0 = floor(xmin), fx1 = ceil(xmax), fy0 = floor(ymin), fy1 = ceil(ymax);
        r[0] = fx0 < 0 ? 0 : (fx0 > W ? W : (int)fx0);
        r[2] = fx1 < 0 ? 0 : (fx1 > W ? W : (int)fx1);
        r[1] = fy0 < 0 ? 0 : (fy0 > H ? H : (int)fy0);
        r[3] = fy1 < 0 ? 0 : (fy1 > H ? H : (int)fy1);
    }
}

/* Launch rectangle: the rendering rectangle grown to the global 8x4 tile grid, so that
 * sub-image rows start on 128-byte boundaries; empty in, empty out. */
VR_HD void vr_launch_rect(const int r[4], int W, int H, int l[4]) {
    if (r[2] <= r[0] || r[3] <= r[1]) {
        l[0] = l[1] = l[2] = l[3] = 0;
        return;
    }
    l[0] = r[0] - (r[0] % VR_TILE_W);
    l[1] = r[1] - (r[1] % VR_TILE_H);
    l[2] = ((r[2] + VR_TILE_W - 1) / VR_TILE_W) * VR_TILE_W;
    l[3] = ((r[3] + VR_TILE_H - 1) / VR_TILE_H) * VR_TILE_H;
    if (l[2] > W) l[2] = W;
    if (l[3] > H) l[3] = H;
}

#endif
