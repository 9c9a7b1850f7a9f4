/*
 * vr_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, double-precision CPU statement of what the bricked ray-casting hot path
 * of Hassan, Fluke & Barnes (arXiv:1205.0282) computes, written from the paper
 * in the paper's order:
 *   - volume split into sub-cubes ("bricks"), each rendered independently at full output
 *     resolution                                         PAPER.md:105,113,136  (§2.1, §2.3.1)
 *   - per pixel: ray start, direction, intersection with the bounding cube, early exit of
 *     rays that miss, march until the exit point or until the opacity / maximum value is
 *     reached                                            PAPER.md:152          (§2.3.2)
 *   - tri-linear interpolation of the data
 *   - transfer function: value -> colour and opacity, accumulated along the ray
 *                                                         PAPER.md:45           (§1.2)
 *   - MIP as the shipped transfer function, arbitrary compositing order; alpha blending is
 *     associative so sub-images composite in visibility order   PAPER.md:174   (§2.3.3)
 *   - rendering rectangle = screen bounding box of the 8 projected sub-cube vertices
 *                                                         PAPER.md:150, Fig.4 :168
 *   - final colour mapping with the user's colour map
 * The paper gives no formulas; every constant and convention is a documented reading
 * R1..R15 (restated in DESIGN.md "Readings"), plus R16 (row f1: per-brick
 * data range, and the transparent-brick rule built on it) and R18 (the paper's
 * per-ray step, selected with step == 0).
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg
 * may load this. It shares no code with paper_1205_0282_b200/ (the CUDA path); only the
 * seeded input generators (synth/) serve both.
 *
 * Pins (tests/test_oracle_pins.py): homogeneous cube closed form, single-voxel tent MIP,
 * axis-aligned orthographic MIP = column max and ALPHA closed form, 1 brick == N bricks,
 * ERT bound, order independence of MIP, per-ray order within global order, each sample
 * owned once, rectangle conservativeness, step-halving convergence, brute force against an
 * independent numpy renderer; data range: planted extremes incl. ghost-only cells, brute
 * force; transparent bricks: their sub-images are exactly zero. Parity unpinned (pure conventions): R1 row orientation,
 * R11 MIP alpha, R13 form of the relative tolerance. R14 (NaN = blanked voxel: a sample with
 * more than 4e-6 of its weight on NaN voxels is dropped, else the NaN corners are left out) is
 * pinned by closed forms on a homogeneous cube with a blanked slab.
 *
 * Build: gcc -O2 -std=c11 -ffp-contract=off -fopenmp -shared -fPIC (oracle/build.py).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define VRO_ALPHA 0
#define VRO_MIP 1

#define VRO_FLAG_ERT_MARGIN 1   /* a termination test had |A_b - tau| < 1e-5          (R12) */
#define VRO_FLAG_OWNER_MARGIN 2 /* an owner decision within 1e-6 voxel, brick ERT'ed   (R12) */
#define VRO_FLAG_LAST_SAMPLE 4  /* MIP: existence of the last sample is marginal       (R12) */
#define VRO_FLAG_GRAZING 8      /* hit/miss of the volume decided by < 1e-9 voxel      (R10) */
#define VRO_FLAG_NAN_MARGIN 16  /* a sample's NaN weight within a factor 2 of the limit (R14) */
#define VRO_NAN_WEIGHT 4e-6     /* R14: tri-linear weight on NaN corners above which a sample is dropped */

typedef float (*vro_voxel_fn)(const void* ctx, int64_t x, int64_t y, int64_t z);

typedef struct vro_volume {
    int64_t n[3];      /* nx, ny, nz */
    int brick, ghost;
    int g[3];          /* grid of bricks */
    int nbricks;
    float** bricks;    /* dense mode: the oracle's own ghost-padded copies */
    vro_voxel_fn fn;   /* procedural mode */
    const void* ctx;
    int ntf;
    float* tf;         /* ntf x 4 straight-alpha RGBA */
    double vmin, vmax;
    double tau;        /* early ray termination threshold; > 1 disables */
    int* order_override; /* test hook: composite in this order instead of R9's */
    int64_t ghost_violations; /* fetches that left the padded brick (R3) */
    double ert_margin; /* R12: a termination test with |A_b - tau| below this flags the pixel (1e-5; the tests of the
                        * texture sampler, whose 8-bit filter weights move A_b by ~1e-4, widen it) */
    double nan_limit;  /* R14: tri-linear weight on NaN corners above which a sample is dropped (VRO_NAN_WEIGHT); the
                        * tests move it by a factor 2 either way to obtain BOTH correct values of a flagged pixel (R12) */
} vro_volume;

/* ------------------------------------------------------------------ bricks (R3, a1) */
static void brick_coords(const vro_volume* v, int b, int bc[3]) {
    bc[0] = b % v->g[0];
    bc[1] = (b / v->g[0]) % v->g[1];
    bc[2] = b / (v->g[0] * v->g[1]);
}
static void brick_core(const vro_volume* v, int b, int64_t lo[3], int64_t hi[3]) {
    int bc[3];
    brick_coords(v, b, bc);
    for (int a = 0; a < 3; ++a) {
        lo[a] = (int64_t)bc[a] * v->brick;
        hi[a] = lo[a] + v->brick;
        if (hi[a] > v->n[a]) hi[a] = v->n[a];
    }
}
static int64_t clamp64(int64_t x, int64_t lo, int64_t hi) { return x < lo ? lo : (x > hi ? hi : x); }

vro_volume* vro_create(int64_t nx, int64_t ny, int64_t nz, int brick, int ghost) {
    if (nx <= 0 || ny <= 0 || nz <= 0 || brick < 2 || ghost < 0) return NULL;
    vro_volume* v = (vro_volume*)calloc(1, sizeof(vro_volume));
    v->n[0] = nx; v->n[1] = ny; v->n[2] = nz;
    v->brick = brick; v->ghost = ghost;
    for (int a = 0; a < 3; ++a) v->g[a] = (int)((v->n[a] + brick - 1) / brick);
    v->nbricks = v->g[0] * v->g[1] * v->g[2];
    v->tau = 0.99;
    v->nan_limit = VRO_NAN_WEIGHT;
    v->ert_margin = 1e-5;
    return v;
}

/* Dense mode: build every brick's ghost-padded copy, edge-replicated at the volume boundary. */
int vro_set_dense(vro_volume* v, const float* src /* [nz][ny][nx] */) {
    if (!v || !src) return 1;
    v->bricks = (float**)calloc((size_t)v->nbricks, sizeof(float*));
    const int g = v->ghost;
    for (int b = 0; b < v->nbricks; ++b) {
        int64_t lo[3], hi[3];
        brick_core(v, b, lo, hi);
        int64_t d0 = hi[0] - lo[0] + 2 * g, d1 = hi[1] - lo[1] + 2 * g, d2 = hi[2] - lo[2] + 2 * g;
        float* p = (float*)malloc((size_t)(d0 * d1 * d2) * sizeof(float));
        if (!p) return 2;
        for (int64_t k = 0; k < d2; ++k) {
            int64_t z = clamp64(lo[2] - g + k, 0, v->n[2] - 1);
            for (int64_t j = 0; j < d1; ++j) {
                int64_t y = clamp64(lo[1] - g + j, 0, v->n[1] - 1);
                for (int64_t i = 0; i < d0; ++i) {
                    int64_t x = clamp64(lo[0] - g + i, 0, v->n[0] - 1);
                    p[(k * d1 + j) * d0 + i] = src[(z * v->n[1] + y) * v->n[0] + x];
                }
            }
        }
        v->bricks[b] = p;
    }
    return 0;
}

int vro_set_procedural(vro_volume* v, vro_voxel_fn fn, const void* ctx) {
    if (!v || !fn) return 1;
    v->fn = fn; v->ctx = ctx;
    return 0;
}

void vro_destroy(vro_volume* v) {
    if (!v) return;
    if (v->bricks) {
        for (int b = 0; b < v->nbricks; ++b) free(v->bricks[b]);
        free(v->bricks);
    }
    free(v->tf);
    free(v->order_override);
    free(v);
}

int vro_num_bricks(const vro_volume* v) { return v->nbricks; }
int64_t vro_ghost_violations(const vro_volume* v) { return v->ghost_violations; }

/* test access to the padded copy of brick b: dims out, pointer returned (dense mode) */
const float* vro_brick_data(const vro_volume* v, int b, int64_t dims[3]) {
    int64_t lo[3], hi[3];
    brick_core(v, b, lo, hi);
    for (int a = 0; a < 3; ++a) dims[a] = hi[a] - lo[a] + 2 * v->ghost;
    return v->bricks ? v->bricks[b] : NULL;
}

/* ------------------------------------------------------------------ data range (row f1)
 * PAPER.md:146 (sec. 2.3.1): "An independent task to determine the local minimum and maximum
 * starts when the data is loaded into the GPU memory"; :152 the march may stop at "the
 * maximum pixel value (defined by the global maximum of the data)".
 * Local = per brick, over the brick's own ghost-padded copy (every value a sample of that
 * brick can interpolate between); b < 0: over all bricks = the range of the whole volume
 * (ghost cells are copies of voxels). Plain loops over the cells. */
int vro_brick_minmax(const vro_volume* v, int b, float* mn_out, float* mx_out) {
    if (!v || b >= v->nbricks || (!v->bricks && !v->fn)) return 1;
    float mn = INFINITY, mx = -INFINITY;
    const int b0 = b < 0 ? 0 : b, b1 = b < 0 ? v->nbricks : b + 1;
    const int g = v->ghost;
    for (int q = b0; q < b1; ++q) {
        int64_t lo[3], hi[3];
        brick_core(v, q, lo, hi);
        const int64_t d0 = hi[0] - lo[0] + 2 * g, d1 = hi[1] - lo[1] + 2 * g, d2 = hi[2] - lo[2] + 2 * g;
        for (int64_t k = 0; k < d2; ++k)
            for (int64_t j = 0; j < d1; ++j)
                for (int64_t i = 0; i < d0; ++i) {
                    float x;
                    if (v->bricks) x = v->bricks[q][(k * d1 + j) * d0 + i];
                    else x = v->fn(v->ctx, clamp64(lo[0] - g + i, 0, v->n[0] - 1), clamp64(lo[1] - g + j, 0, v->n[1] - 1),
                                   clamp64(lo[2] - g + k, 0, v->n[2] - 1));
                    if (x < mn) mn = x;
                    if (x > mx) mx = x;
                }
    }
    *mn_out = mn;
    *mx_out = mx;
    return 0;
}

/* R16: a brick is TRANSPARENT for the current transfer function - and may be skipped in ALPHA
 * mode without changing a single output bit - iff every table entry a sample of the brick can
 * interpolate between has alpha == 0. The entry range is an integer decision taken in
 * float32 (the precision the kernel classifies in), widened by one entry below and two above
 * so that a rounding of the interpolated value cannot leave it:
 *   I(x) = min(floor(sat((x - vmin) * inv_range) * (n-1)), n-2),  inv_range = (float)(1/(vmax-vmin))
 *   transparent <=> a_i == 0 for all i in [max(0, I(min_b) - 1), min(n-1, I(max_b) + 2)].  */
static int tf_index_f32(const vro_volume* v, float x) {
    const float vminf = (float)v->vmin;
    const float inv_range = (float)(1.0 / ((double)(float)v->vmax - (double)(float)v->vmin));
    float u = (x - vminf) * inv_range;
    if (!(u > 0.0f)) u = 0.0f;
    if (u > 1.0f) u = 1.0f;
    const float t = u * (float)(v->ntf - 1);
    int i = (int)t;
    if (i > v->ntf - 2) i = v->ntf - 2;
    return i;
}
int vro_brick_transparent(const vro_volume* v, int b) {
    float mn, mx;
    if (!v || !v->tf || b < 0 || vro_brick_minmax(v, b, &mn, &mx)) return -1;
    int i0 = tf_index_f32(v, mn) - 1, i1 = tf_index_f32(v, mx) + 2;
    if (i0 < 0) i0 = 0;
    if (i1 > v->ntf - 1) i1 = v->ntf - 1;
    for (int i = i0; i <= i1; ++i)
        if (v->tf[4 * i + 3] != 0.0f) return 0;
    return 1;
}

int vro_set_tf(vro_volume* v, const float* rgba, int n, double vmin, double vmax) {
    if (!v || !rgba || n < 2 || !(vmax > vmin)) return 1;
    for (int i = 0; i < n; ++i) /* R7: the table's alpha is an opacity per voxel of path, 1 - (1-a)^w needs a in [0,1] */
        if (!(rgba[4 * i + 3] >= 0.0f && rgba[4 * i + 3] <= 1.0f)) return 1;
    free(v->tf);
    v->tf = (float*)malloc((size_t)n * 4 * sizeof(float));
    memcpy(v->tf, rgba, (size_t)n * 4 * sizeof(float));
    v->ntf = n; v->vmin = vmin; v->vmax = vmax;
    return 0;
}
void vro_set_tau(vro_volume* v, double tau) { v->tau = tau; }
/* R12/R14 test hook: the drop limit of R14 scaled by `scale` (1 = the reading's 4e-6). The NAN_MARGIN flag keeps
 * marking samples within a factor 2 of the NOMINAL limit, so scale 0.5 drops and scale 2 keeps every flagged sample. */
/* R12 test hook: width of the band around tau inside which a termination test flags its pixel (default 1e-5). */
void vro_set_ert_margin(vro_volume* v, double margin) { v->ert_margin = margin; }
void vro_set_nan_limit_scale(vro_volume* v, double scale) { v->nan_limit = VRO_NAN_WEIGHT * scale; }
int vro_set_order_override(vro_volume* v, const int* order) {
    free(v->order_override);
    v->order_override = NULL;
    if (order) {
        v->order_override = (int*)malloc((size_t)v->nbricks * sizeof(int));
        memcpy(v->order_override, order, (size_t)v->nbricks * sizeof(int));
    }
    return 0;
}

/* Voxel (ix,iy,iz) in GLOBAL index space as seen by brick b (R3): read from the brick's own
 * padded copy; a fetch outside the padded extent is clamped into it and counted. */
static double brick_voxel(vro_volume* v, int b, const int64_t lo[3], const int64_t hi[3], int64_t ix, int64_t iy, int64_t iz) {
    const int g = v->ghost;
    int64_t d0 = hi[0] - lo[0] + 2 * g, d1 = hi[1] - lo[1] + 2 * g, d2 = hi[2] - lo[2] + 2 * g;
    int64_t i = ix - (lo[0] - g), j = iy - (lo[1] - g), k = iz - (lo[2] - g);
    if (i < 0 || i >= d0 || j < 0 || j >= d1 || k < 0 || k >= d2) {
#pragma omp atomic
        v->ghost_violations++;
        i = clamp64(i, 0, d0 - 1); j = clamp64(j, 0, d1 - 1); k = clamp64(k, 0, d2 - 1);
    }
    if (v->bricks) return (double)v->bricks[b][(k * d1 + j) * d0 + i];
    /* procedural: the padded cell's content is the edge-replicated global voxel */
    return (double)v->fn(v->ctx, clamp64(lo[0] - g + i, 0, v->n[0] - 1), clamp64(lo[1] - g + j, 0, v->n[1] - 1),
                         clamp64(lo[2] - g + k, 0, v->n[2] - 1));
}

/* R3: voxel (i,j,k) is centred at (i+1/2, j+1/2, k+1/2); tri-linear interpolation. */
static double trilinear(vro_volume* v, int b, const int64_t lo[3], const int64_t hi[3], const double p[3], double* nan_weight) {
    int64_t i0[3];
    double f[3];
    for (int a = 0; a < 3; ++a) {
        double q = p[a] - 0.5;
        double fl = floor(q);
        i0[a] = (int64_t)fl;
        f[a] = q - fl;
    }
    double c[2][2][2];
    for (int dz = 0; dz < 2; ++dz)
        for (int dy = 0; dy < 2; ++dy)
            for (int dx = 0; dx < 2; ++dx) c[dz][dy][dx] = brick_voxel(v, b, lo, hi, i0[0] + dx, i0[1] + dy, i0[2] + dz);
    double c00 = c[0][0][0] + f[0] * (c[0][0][1] - c[0][0][0]);
    double c01 = c[0][1][0] + f[0] * (c[0][1][1] - c[0][1][0]);
    double c10 = c[1][0][0] + f[0] * (c[1][0][1] - c[1][0][0]);
    double c11 = c[1][1][0] + f[0] * (c[1][1][1] - c[1][1][0]);
    double c0 = c00 + f[1] * (c01 - c00);
    double c1 = c10 + f[1] * (c11 - c10);
    double val = c0 + f[2] * (c1 - c0);
    if (nan_weight) *nan_weight = 0.0;
    if (isnan(val)) {
        /* R14: blanked (NaN) voxels. N = the tri-linear weight that falls on NaN corners. N > 4e-6: the
         * sample is dropped (NaN returned). Otherwise the NaN corners are left out and the rest
         * renormalised: val = sum over valid corners of w_i v_i / (1 - N) - continuous where a sample sits
         * on a cell boundary and a NaN neighbour has weight 0 (the paper's per-ray step puts whole rays there). */
        double N = 0.0, acc = 0.0;
        for (int dz = 0; dz < 2; ++dz)
            for (int dy = 0; dy < 2; ++dy)
                for (int dx = 0; dx < 2; ++dx) {
                    double w = (dx ? f[0] : 1.0 - f[0]) * (dy ? f[1] : 1.0 - f[1]) * (dz ? f[2] : 1.0 - f[2]);
                    if (isnan(c[dz][dy][dx])) N += w;
                    else acc += w * c[dz][dy][dx];
                }
        if (nan_weight) *nan_weight = N;
        val = (N > v->nan_limit) ? NAN : acc / (1.0 - N);
    }
    return val;
}

/* ------------------------------------------------------------------ view (R1, R2, R9) */
typedef struct {
    double M[16], Minv[16]; /* column-major, clip = M * world */
    int ortho;
    double eye[3];          /* perspective: eye point; orthographic: forward direction */
} vro_view;

static void mat_mul(const double* A, const double* B, double* C) { /* C = A*B, column-major */
    for (int c = 0; c < 4; ++c)
        for (int r = 0; r < 4; ++r) {
            double s = 0.0;
            for (int k = 0; k < 4; ++k) s += A[k * 4 + r] * B[c * 4 + k];
            C[c * 4 + r] = s;
        }
}

static int mat_inv(const double* A, double* Ainv) { /* Gauss-Jordan, partial pivoting */
    double a[4][8];
    for (int r = 0; r < 4; ++r)
        for (int c = 0; c < 4; ++c) { a[r][c] = A[c * 4 + r]; a[r][4 + c] = (r == c) ? 1.0 : 0.0; }
    for (int col = 0; col < 4; ++col) {
        int piv = col;
        for (int r = col + 1; r < 4; ++r) if (fabs(a[r][col]) > fabs(a[piv][col])) piv = r;
        if (a[piv][col] == 0.0) return 1;
        if (piv != col) for (int c = 0; c < 8; ++c) { double t = a[piv][c]; a[piv][c] = a[col][c]; a[col][c] = t; }
        double d = a[col][col];
        for (int c = 0; c < 8; ++c) a[col][c] /= d;
        for (int r = 0; r < 4; ++r) if (r != col) {
            double f = a[r][col];
            if (f != 0.0) for (int c = 0; c < 8; ++c) a[r][c] -= f * a[col][c];
        }
    }
    for (int r = 0; r < 4; ++r) for (int c = 0; c < 4; ++c) Ainv[c * 4 + r] = a[r][4 + c];
    return 0;
}

static void mat_vec(const double* A, const double x[4], double y[4]) {
    for (int r = 0; r < 4; ++r) y[r] = A[0 + r] * x[0] + A[4 + r] * x[1] + A[8 + r] * x[2] + A[12 + r] * x[3];
}

static int view_setup(const float* view, const float* proj, vro_view* vw) {
    double V[16], P[16];
    for (int i = 0; i < 16; ++i) { V[i] = (double)view[i]; P[i] = (double)proj[i]; }
    mat_mul(P, V, vw->M);
    if (mat_inv(vw->M, vw->Minv)) return 1;
    for (int i = 0; i < 16; ++i) if (!isfinite(vw->Minv[i])) return 1;
    /* R9: homogeneous eye = Minv * (0,0,1,0) */
    const double e4[4] = {0.0, 0.0, 1.0, 0.0};
    double c[4];
    mat_vec(vw->Minv, e4, c);
    double mag = fabs(c[0]) + fabs(c[1]) + fabs(c[2]);
    if (fabs(c[3]) < 1e-9 * mag) {
        vw->ortho = 1;
        for (int a = 0; a < 3; ++a) vw->eye[a] = c[a];
    } else {
        vw->ortho = 0;
        for (int a = 0; a < 3; ++a) vw->eye[a] = c[a] / c[3];
    }
    return 0;
}

static void unproject(const vro_view* vw, double x, double y, double z, double out[3]) {
    const double c[4] = {x, y, z, 1.0};
    double p[4];
    mat_vec(vw->Minv, c, p);
    for (int a = 0; a < 3; ++a) out[a] = p[a] / p[3];
}

/* R1, R2: pixel (i,j), row 0 at the bottom, centres at half-integers; ray from the near
 * plane to the far plane. Returns t_far. */
static double pixel_ray(const vro_view* vw, int W, int H, int i, int j, double o[3], double d[3]) {
    double x = 2.0 * ((double)i + 0.5) / (double)W - 1.0;
    double y = 2.0 * ((double)j + 0.5) / (double)H - 1.0;
    double nr[3], fr[3];
    unproject(vw, x, y, -1.0, nr);
    unproject(vw, x, y, 1.0, fr);
    double len = 0.0;
    for (int a = 0; a < 3; ++a) { d[a] = fr[a] - nr[a]; len += d[a] * d[a]; }
    len = sqrt(len);
    for (int a = 0; a < 3; ++a) { d[a] /= len; o[a] = nr[a]; }
    return len;
}

/* R4: slab test of (o,d) against the half-open box [lo,hi) (closed where `closed_hi[a]`).
 * Returns 1 and [tin,tout] if the line meets the box; margin = smallest decision margin. */
static int slab(const double o[3], const double d[3], const double lo[3], const double hi[3], const int closed_hi[3],
                double* tin, double* tout, double* margin) {
    double t0 = -INFINITY, t1 = INFINITY, mg = INFINITY;
    for (int a = 0; a < 3; ++a) {
        if (d[a] == 0.0) {
            int inside = (o[a] >= lo[a]) && (closed_hi[a] ? (o[a] <= hi[a]) : (o[a] < hi[a]));
            double m = fmin(fabs(o[a] - lo[a]), fabs(o[a] - hi[a]));
            if (m < mg) mg = m;
            if (!inside) { *margin = mg; return 0; }
        } else {
            double ta = (lo[a] - o[a]) / d[a], tb = (hi[a] - o[a]) / d[a];
            if (ta > tb) { double t = ta; ta = tb; tb = t; }
            if (ta > t0) t0 = ta;
            if (tb < t1) t1 = tb;
        }
    }
    *tin = t0; *tout = t1;
    double m = fabs(t1 - t0);
    if (m < mg) mg = m;
    *margin = mg;
    return t1 >= t0;
}

/* ------------------------------------------------------------------ visibility order (R9, a3) */
static void axis_ranks(const vro_volume* v, const vro_view* vw, int a, int* rank) {
    int n = v->g[a];
    if (vw->ortho) {
        for (int i = 0; i < n; ++i) rank[i] = (vw->eye[a] >= 0.0) ? i : (n - 1 - i);
        return;
    }
    double* dist = (double*)malloc((size_t)n * sizeof(double));
    for (int i = 0; i < n; ++i) {
        double lo = (double)i * v->brick, hi = lo + v->brick;
        if (hi > (double)v->n[a]) hi = (double)v->n[a];
        double e = vw->eye[a];
        dist[i] = (e < lo) ? (lo - e) : ((e > hi) ? (e - hi) : 0.0);
    }
    for (int i = 0; i < n; ++i) {
        int r = 0;
        for (int j = 0; j < n; ++j) if (dist[j] < dist[i] || (dist[j] == dist[i] && j < i)) ++r;
        rank[i] = r;
    }
    free(dist);
}

static void brick_order(const vro_volume* v, const vro_view* vw, int* order /* front to back */) {
    if (v->order_override) { memcpy(order, v->order_override, (size_t)v->nbricks * sizeof(int)); return; }
    int* rk[3];
    for (int a = 0; a < 3; ++a) { rk[a] = (int*)malloc((size_t)v->g[a] * sizeof(int)); axis_ranks(v, vw, a, rk[a]); }
    /* key = (rank_z, rank_y, rank_x) lexicographic; ranks are permutations so keys are unique */
    for (int b = 0; b < v->nbricks; ++b) {
        int bc[3];
        brick_coords(v, b, bc);
        int key = (rk[2][bc[2]] * v->g[1] + rk[1][bc[1]]) * v->g[0] + rk[0][bc[0]];
        order[key] = b;
    }
    for (int a = 0; a < 3; ++a) free(rk[a]);
}

int vro_brick_order(vro_volume* v, const float* view, const float* proj, int* order) {
    vro_view vw;
    if (view_setup(view, proj, &vw)) return 1;
    brick_order(v, &vw, order);
    return 0;
}

/* ------------------------------------------------------------------ rendering rectangle (a2) */
/* project the 8 sub-cube vertices, take the bounding rectangle. Half-open
 * pixel ranges [x0,x1) x [y0,y1), clipped to the viewport; a vertex with clip w <= 0 makes
 * the rectangle the whole viewport (conservative). */
int vro_rects(vro_volume* v, const float* view, const float* proj, int W, int H, int* rects /* nbricks x 4 */) {
    vro_view vw;
    if (view_setup(view, proj, &vw)) return 1;
    for (int b = 0; b < v->nbricks; ++b) {
        int64_t lo[3], hi[3];
        brick_core(v, b, lo, hi);
        double xmin = INFINITY, xmax = -INFINITY, ymin = INFINITY, ymax = -INFINITY;
        int full = 0;
        for (int c = 0; c < 8; ++c) {
            double w4[4] = {(c & 1) ? (double)hi[0] : (double)lo[0], (c & 2) ? (double)hi[1] : (double)lo[1],
                            (c & 4) ? (double)hi[2] : (double)lo[2], 1.0};
            double q[4];
            mat_vec(vw.M, w4, q);
            if (!(q[3] > 1e-12)) { full = 1; break; }
            double px = (q[0] / q[3] + 1.0) * 0.5 * W, py = (q[1] / q[3] + 1.0) * 0.5 * H;
            if (px < xmin) xmin = px;
            if (px > xmax) xmax = px;
            if (py < ymin) ymin = py;
            if (py > ymax) ymax = py;
        }
        int x0 = 0, y0 = 0, x1 = W, y1 = H;
        if (!full) {
            double fx0 = floor(xmin), fx1 = ceil(xmax), fy0 = floor(ymin), fy1 = ceil(ymax);
            x0 = fx0 < 0 ? 0 : (fx0 > W ? W : (int)fx0);
            x1 = fx1 < 0 ? 0 : (fx1 > W ? W : (int)fx1);
            y0 = fy0 < 0 ? 0 : (fy0 > H ? H : (int)fy0);
            y1 = fy1 < 0 ? 0 : (fy1 > H ? H : (int)fy1);
        }
        rects[4 * b + 0] = x0; rects[4 * b + 1] = y0; rects[4 * b + 2] = x1; rects[4 * b + 3] = y1;
    }
    return 0;
}

/* ------------------------------------------------------------------ classification (R7, a6) */
static void classify(const vro_volume* v, double val, double rgba[4]) {
    double u = (val - v->vmin) / (v->vmax - v->vmin);
    if (u < 0.0) u = 0.0;
    if (u > 1.0) u = 1.0;
    double x = u * (double)(v->ntf - 1);
    int i = (int)floor(x);
    if (i > v->ntf - 2) i = v->ntf - 2;
    double f = x - (double)i;
    for (int c = 0; c < 4; ++c) {
        double a = (double)v->tf[4 * i + c], b = (double)v->tf[4 * (i + 1) + c];
        rgba[c] = a + f * (b - a);
    }
}

/* ------------------------------------------------------------------ one pixel (steps 1-8) */
typedef struct {
    double C[3], A; /* ALPHA: premultiplied colour, opacity */
    double m;       /* MIP: running max */
    int64_t count;  /* samples taken */
    int stopped;
} brick_acc;

static void render_pixel(vro_volume* v, const vro_view* vw, const int* order, int W, int H, int i, int j, double step,
                         int mode, brick_acc* acc, double out[4], uint8_t* flag, int64_t* ntaken, int64_t* nsched,
                         double* sub /* nbricks x 4 or NULL */) {
    const int nb = v->nbricks;
    uint8_t fl = 0;
    out[0] = out[1] = out[2] = out[3] = 0.0;
    for (int b = 0; b < nb; ++b) { acc[b].C[0] = acc[b].C[1] = acc[b].C[2] = acc[b].A = 0.0; acc[b].m = -INFINITY; acc[b].count = 0; acc[b].stopped = 0; }
    int64_t taken = 0, sched = 0;

    /* step 1: the ray */
    double o[3], d[3];
    double tfar = pixel_ray(vw, W, H, i, j, o, d);
    /* step 2: global slab test (R4) */
    const double glo[3] = {0.0, 0.0, 0.0}, ghi[3] = {(double)v->n[0], (double)v->n[1], (double)v->n[2]};
    const int closed[3] = {1, 1, 1};
    double tin, tout, mg;
    int hit = slab(o, d, glo, ghi, closed, &tin, &tout, &mg);
    double t0 = 0.0, t1 = 0.0;
    if (hit) {
        t0 = tin > 0.0 ? tin : 0.0;
        t1 = tout < tfar ? tout : tfar;
        if (!(t1 > t0)) hit = 0;
        if (fabs(t1 - t0) < 1e-9) fl |= VRO_FLAG_GRAZING;
    }
    if (mg < 1e-9) fl |= VRO_FLAG_GRAZING;
    if (hit) {
        /* R18 (row f2 (i)): step == 0 asks for the paper's per-ray step, "a discrete ray-casting with
         * at least one sample for each voxel intersected" (after Kaufman): one sample per
         * unit advance along the ray's major axis, step = 1 / max_a |d_a| (d is a unit vector). */
        if (step == 0.0) {
            double m = fabs(d[0]);
            if (fabs(d[1]) > m) m = fabs(d[1]);
            if (fabs(d[2]) > m) m = fabs(d[2]);
            step = 1.0 / m;
        }
        /* step 3: sample schedule anchored at the global entry (R5) */
        int64_t K = (int64_t)ceil((t1 - t0) / step);
        double min_owner_margin = INFINITY;
        int any_stopped = 0;
        for (int64_t k = 0; k < K; ++k) {
            double a0 = t0 + (double)k * step, a1 = t0 + (double)(k + 1) * step;
            if (a1 > t1) a1 = t1;
            double w = a1 - a0;
            if (!(w > 0.0)) continue;
            ++sched;
            if (k == K - 1 && mode == VRO_MIP && (w < 1e-6 || step - w < 1e-6)) fl |= VRO_FLAG_LAST_SAMPLE;
            double s = 0.5 * (a0 + a1);
            double p[3];
            for (int a = 0; a < 3; ++a) p[a] = fma(s, d[a], o[a]);
            /* step 4: owner brick by position in half-open core boxes (R6) */
            int bc[3];
            for (int a = 0; a < 3; ++a) {
                double q = p[a] / (double)v->brick;
                int c = (int)floor(q);
                if (c < 0) c = 0;
                if (c > v->g[a] - 1) c = v->g[a] - 1;
                bc[a] = c;
                double r = p[a] - floor(q) * (double)v->brick; /* distance above the lower face */
                double m2 = fmin(r, (double)v->brick - r);
                if (m2 < min_owner_margin) min_owner_margin = m2;
            }
            int b = (bc[2] * v->g[1] + bc[1]) * v->g[0] + bc[0];
            brick_acc* B = &acc[b];
            if (mode == VRO_ALPHA) {
                /* step 7: brick-local early ray termination, tested before the sample (R8) */
                if (B->stopped) continue;
                if (fabs(B->A - v->tau) < v->ert_margin) fl |= VRO_FLAG_ERT_MARGIN;
                if (B->A >= v->tau) { B->stopped = 1; any_stopped = 1; continue; }
            }
            /* step 5: value from the brick's own padded copy (R3) */
            int64_t lo[3], hi[3];
            brick_core(v, b, lo, hi);
            double nanw;
            double val = trilinear(v, b, lo, hi, p, &nanw);
            /* R14: blanked voxels are NaN (the usual convention of radio cubes). A sample with more than
             * 4e-6 of its tri-linear weight on NaN voxels is dropped: it is not taken, adds nothing in
             * ALPHA and cannot be the maximum in MIP. */
            if (nanw > 0.5 * VRO_NAN_WEIGHT && nanw < 2.0 * VRO_NAN_WEIGHT) fl |= VRO_FLAG_NAN_MARGIN;
            if (isnan(val)) continue;
            B->count++;
            ++taken;
            if (mode == VRO_MIP) {
                if (val > B->m) B->m = val;
            } else {
                /* step 6: classify, opacity for a path of length w (R7) */
                double rgba[4];
                classify(v, val, rgba);
                double alpha = 1.0 - pow(1.0 - rgba[3], w);
                double tr = 1.0 - B->A;
                for (int c = 0; c < 3; ++c) B->C[c] += tr * alpha * rgba[c];
                B->A += tr * alpha;
            }
        }
        if (min_owner_margin < 1e-6 && any_stopped) fl |= VRO_FLAG_OWNER_MARGIN;
        /* step 8: sort-last compositing in the canonical order (R9, R11) */
        if (mode == VRO_ALPHA) {
            double C[3] = {0.0, 0.0, 0.0}, A = 0.0;
            for (int q = 0; q < nb; ++q) {
                const brick_acc* B = &acc[order[q]];
                for (int c = 0; c < 3; ++c) C[c] += (1.0 - A) * B->C[c];
                A += (1.0 - A) * B->A;
            }
            out[0] = C[0]; out[1] = C[1]; out[2] = C[2]; out[3] = A;
        } else {
            double m = -INFINITY;
            for (int q = 0; q < nb; ++q) if (acc[order[q]].m > m) m = acc[order[q]].m;
            if (taken > 0) {
                double rgba[4];
                classify(v, m, rgba);
                out[0] = rgba[0]; out[1] = rgba[1]; out[2] = rgba[2]; out[3] = 1.0;
            }
        }
    }
    if (sub) {
        for (int b = 0; b < nb; ++b) {
            if (mode == VRO_ALPHA) { sub[4 * b] = acc[b].C[0]; sub[4 * b + 1] = acc[b].C[1]; sub[4 * b + 2] = acc[b].C[2]; sub[4 * b + 3] = acc[b].A; }
            else { sub[4 * b] = acc[b].m; sub[4 * b + 1] = (double)acc[b].count; sub[4 * b + 2] = 0.0; sub[4 * b + 3] = 0.0; }
        }
    }
    *flag = fl; *ntaken = taken; *nsched = sched;
}

/* Render either a full frame (pixels == NULL: out is [H][W][4]) or a list of npix pixels
 * (pixels = (i,j) pairs: out is [npix][4]). flags / counts / sub may be NULL.
 * counts[2*p] = samples taken, counts[2*p+1] = samples scheduled (before ERT). */
int vro_render(vro_volume* v, const float* view, const float* proj, int W, int H, double step, int mode,
               const int* pixels, int64_t npix, double* out, uint8_t* flags, int64_t* counts, double* sub, int nthreads) {
    if (!v || !view || !proj || W <= 0 || H <= 0 || !(step >= 0.0) || !out) return 1;
    if (mode != VRO_ALPHA && mode != VRO_MIP) return 1;
    if (!v->tf) return 3;
    if (!v->bricks && !v->fn) return 3;
    vro_view vw;
    if (view_setup(view, proj, &vw)) return 2;
    int* order = (int*)malloc((size_t)v->nbricks * sizeof(int));
    brick_order(v, &vw, order);
    int64_t n = pixels ? npix : (int64_t)W * H;
    if (nthreads < 1) nthreads = 1;
#pragma omp parallel num_threads(nthreads)
    {
        brick_acc* acc = (brick_acc*)malloc((size_t)v->nbricks * sizeof(brick_acc));
#pragma omp for schedule(dynamic, 64)
        for (int64_t q = 0; q < n; ++q) {
            int i = pixels ? pixels[2 * q] : (int)(q % W);
            int j = pixels ? pixels[2 * q + 1] : (int)(q / W);
            uint8_t fl;
            int64_t tk, sc;
            render_pixel(v, &vw, order, W, H, i, j, step, mode, acc, out + 4 * q, &fl, &tk, &sc,
                         sub ? sub + (size_t)q * 4 * v->nbricks : NULL);
            if (flags) flags[q] = fl;
            if (counts) { counts[2 * q] = tk; counts[2 * q + 1] = sc; }
        }
        free(acc);
    }
    free(order);
    return 0;
}

/* ------------------------------------------------------------------ ray-brick lists (R10) */
/* Per pixel: bricks whose core box overlaps [t0,t1] with positive length, by increasing
 * t_in. counts[p] = length (<= maxlen written), grazing[p] = 1 if any margin < 1e-9. */
int vro_ray_bricks(vro_volume* v, const float* view, const float* proj, int W, int H, const int* pixels, int64_t npix,
                   int* counts, int* lists, int maxlen, uint8_t* grazing) {
    vro_view vw;
    if (view_setup(view, proj, &vw)) return 2;
    const double glo[3] = {0.0, 0.0, 0.0}, ghi[3] = {(double)v->n[0], (double)v->n[1], (double)v->n[2]};
    const int closed[3] = {1, 1, 1};
    double* tins = (double*)malloc((size_t)v->nbricks * sizeof(double));
    int* ids = (int*)malloc((size_t)v->nbricks * sizeof(int));
    for (int64_t q = 0; q < npix; ++q) {
        double o[3], d[3];
        double tfar = pixel_ray(&vw, W, H, pixels[2 * q], pixels[2 * q + 1], o, d);
        double tin, tout, mg;
        int gz = 0, cnt = 0;
        int hit = slab(o, d, glo, ghi, closed, &tin, &tout, &mg);
        if (mg < 1e-9) gz = 1;
        double t0 = tin > 0.0 ? tin : 0.0, t1 = tout < tfar ? tout : tfar;
        if (hit && t1 > t0) {
            for (int b = 0; b < v->nbricks; ++b) {
                int64_t lo[3], hi[3];
                brick_core(v, b, lo, hi);
                double blo[3], bhi[3];
                int bcl[3];
                for (int a = 0; a < 3; ++a) { blo[a] = (double)lo[a]; bhi[a] = (double)hi[a]; bcl[a] = (hi[a] == v->n[a]); }
                double bi, bo, bm;
                int bh = slab(o, d, blo, bhi, bcl, &bi, &bo, &bm);
                if (!bh) { if (bm < 1e-9) gz = 1; continue; }
                double a0 = bi > t0 ? bi : t0, a1 = bo < t1 ? bo : t1;
                if (fabs(a1 - a0) < 1e-9) gz = 1;
                if (a1 > a0) { tins[cnt] = a0; ids[cnt] = b; ++cnt; }
            }
            for (int x = 1; x < cnt; ++x) { /* insertion sort by t_in */
                double tv = tins[x]; int iv = ids[x]; int y = x - 1;
                while (y >= 0 && tins[y] > tv) { tins[y + 1] = tins[y]; ids[y + 1] = ids[y]; --y; }
                tins[y + 1] = tv; ids[y + 1] = iv;
            }
            for (int x = 1; x < cnt; ++x) if (fabs(tins[x] - tins[x - 1]) < 1e-9) gz = 1;
        }
        counts[q] = cnt;
        for (int x = 0; x < cnt && x < maxlen; ++x) lists[q * maxlen + x] = ids[x];
        if (grazing) grazing[q] = (uint8_t)gz;
    }
    free(tins); free(ids);
    return 0;
}

/* ------------------------------------------------------------------ standalone compositing (R15, a9) */
/* layers[l] is a premultiplied RGBA float32 sub-image covering rects[l] = (x0,y0,x1,y1),
 * stored [y1-y0][x1-x0][4]. Front-to-back `over` in the given order, in double. */
int vro_composite(const float* const* layers, const int* rects, const int* order, int n, int W, int H,
                  const int* pixels, int64_t npix, double* out, int nthreads) {
    int64_t np_ = pixels ? npix : (int64_t)W * H;
    if (nthreads < 1) nthreads = 1;
#pragma omp parallel for num_threads(nthreads) schedule(static)
    for (int64_t q = 0; q < np_; ++q) {
        int i = pixels ? pixels[2 * q] : (int)(q % W);
        int j = pixels ? pixels[2 * q + 1] : (int)(q / W);
        double C[3] = {0.0, 0.0, 0.0}, A = 0.0;
        for (int s = 0; s < n; ++s) {
            int l = order[s];
            const int* r = rects + 4 * l;
            if (i < r[0] || i >= r[2] || j < r[1] || j >= r[3]) continue;
            const float* px = layers[l] + ((int64_t)(j - r[1]) * (r[2] - r[0]) + (i - r[0])) * 4;
            for (int c = 0; c < 3; ++c) C[c] += (1.0 - A) * (double)px[c];
            A += (1.0 - A) * (double)px[3];
        }
        out[4 * q] = C[0]; out[4 * q + 1] = C[1]; out[4 * q + 2] = C[2]; out[4 * q + 3] = A;
    }
    return 0;
}
