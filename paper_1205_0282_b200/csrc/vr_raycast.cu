/*
 * vr_raycast.cu -- the per-brick ray-cast kernel.
 *
 * PAPER.md:152 (sec. 2.3.2): each GPU thread computes its ray's start and direction and its
 * intersection with the bounding cube, rays that miss leave at once, the ray is marched until
 * the exit point or until the opacity / the maximum value is reached; :69,:150 tri-linear
 * interpolation of the data; :45 transfer function -> colour and opacity accumulated along
 * the ray; :174 MIP. One thread = one pixel of one brick's rendering rectangle (:150).
 *
 * B200 design:
 *   - persistent grid (resident CTAs x 148 SMs); warps pull (brick, 8x4-pixel tile) work items
 *     from a device-built list with one atomic per item, bricks in visibility order so the
 *     tiles in flight share one or two bricks in L2;
 *   - ray, global clip and the integer sample range each brick owns are computed once per
 *     (ray, brick) in FP64 with individually rounded operations, so the kernel takes exactly
 *     the sample set the definition prescribes (R5, R6);
 *   - sample positions advance on a 32.32 fixed-point lattice in brick-local coordinates
 *     (two integer adds per axis and step): the integer word is the voxel index, the fraction
 *     word becomes the float32 interpolation weight with a shift/or - no FP64 and no
 *     int<->float conversion in the loop, and a position error below 1e-7 voxel;
 *   - tri-linear interpolation is hand-rolled in float32 on 8 read-only loads (hardware
 *     texture filtering has 8-bit weights and cannot meet the MIP tolerance);
 *   - the LUT is staged in shared memory as (entry, delta) pairs;
 *   - early ray termination and loop exit are warp votes.
 */
#include <limits.h>

#include "vr_view.cuh"

#define FULL_MASK 0xffffffffu
#ifndef VR_REUSE
#define VR_REUSE 1 /* keep the 8 voxels while consecutive samples stay in the same cell */
#endif
#ifndef VR_RECOMPUTE_TAIL
#define VR_RECOMPUTE_TAIL 1 /* rebuild the FP64 ray for the exit samples instead of keeping it live */
#endif
#ifndef VR_MIN_CTAS
#define VR_MIN_CTAS 3 /* resident CTAs per SM the register budget is cut for (80 registers) */
#endif

struct RaySetup {
    double o[3], d[3];
    double t0, t1;
    int K; /* number of scheduled samples; 0 = miss */
};

/* R1, R2: pixel (i,j), centres at half-integers, row 0 at the bottom; ray from the near plane
 * (clip z = -1) to the far plane (+1). R4: slab test against the closed global box. */
__device__ __forceinline__ void ray_setup(const double* __restrict__ Minv, int W, int H, int i, int j, const VrGrid& g,
                                          double step, RaySetup& r) {
    const double x = VR_SUB(VR_DIV(VR_MUL(2.0, VR_ADD((double)i, 0.5)), (double)W), 1.0);
    const double y = VR_SUB(VR_DIV(VR_MUL(2.0, VR_ADD((double)j, 0.5)), (double)H), 1.0);
    double nr[4], fr[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const double xy = VR_ADD(VR_MUL(Minv[k], x), VR_MUL(Minv[4 + k], y));
        const double w = VR_MUL(Minv[12 + k], 1.0);
        nr[k] = VR_ADD(VR_ADD(xy, VR_MUL(Minv[8 + k], -1.0)), w);
        fr[k] = VR_ADD(VR_ADD(xy, VR_MUL(Minv[8 + k], 1.0)), w);
    }
    double len = 0.0;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        const double na = VR_DIV(nr[a], nr[3]);
        const double fa = VR_DIV(fr[a], fr[3]);
        r.o[a] = na;
        r.d[a] = VR_SUB(fa, na);
        len = VR_ADD(len, VR_MUL(r.d[a], r.d[a]));
    }
    len = VR_SQRT(len);
#pragma unroll
    for (int a = 0; a < 3; ++a) r.d[a] = VR_DIV(r.d[a], len);
    const double tfar = len;

    double tin = -INFINITY, tout = INFINITY;
    bool hit = true;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        const double hi = (double)g.n[a];
        if (r.d[a] == 0.0) {
            if (!(r.o[a] >= 0.0 && r.o[a] <= hi)) hit = false;
        } else {
            double ta = VR_DIV(VR_SUB(0.0, r.o[a]), r.d[a]);
            double tb = VR_DIV(VR_SUB(hi, r.o[a]), r.d[a]);
            if (ta > tb) {
                const double t = ta;
                ta = tb;
                tb = t;
            }
            if (ta > tin) tin = ta;
            if (tb < tout) tout = tb;
        }
    }
    r.K = 0;
    r.t0 = 0.0;
    r.t1 = 0.0;
    if (hit && tout >= tin) {
        const double t0 = tin > 0.0 ? tin : 0.0;
        const double t1 = tout < tfar ? tout : tfar;
        if (t1 > t0) {
            r.t0 = t0;
            r.t1 = t1;
            const double kd = ceil(VR_DIV(VR_SUB(t1, t0), step));
            r.K = kd > 1073741824.0 ? 1073741824 : (int)kd;
        }
    }
}

/* R5: sample k stands for the interval [t0 + k step, min(t0 + (k+1) step, t1)]: s = its
 * midpoint, w = its length; intervals of non-positive length are dropped. */
__device__ __forceinline__ bool sample_sw(const RaySetup& r, double step, int k, double& s, double& w) {
    const double a0 = VR_ADD(r.t0, VR_MUL((double)k, step));
    double a1 = VR_ADD(r.t0, VR_MUL((double)(k + 1), step));
    if (a1 > r.t1) a1 = r.t1;
    w = VR_SUB(a1, a0);
    s = VR_MUL(0.5, VR_ADD(a0, a1));
    return w > 0.0;
}

/* R6: owner of sample k along axis a = clamp(floor(p_a / brick), 0, g_a - 1), p = o + s d. */
__device__ __forceinline__ int owner_axis(const RaySetup& r, const VrGrid& g, double s, int a) {
    const double p = VR_FMA(s, r.d[a], r.o[a]);
    const double q = g.brick_pow2 ? VR_MUL(p, 1.0 / (double)g.brick) : VR_DIV(p, (double)g.brick);
    const double f = floor(q);
    int c = (f < 0.0) ? 0 : ((f > (double)(g.g[a] - 1)) ? g.g[a] - 1 : (int)f);
    return c;
}

/* Monotone predicates in k (each axis coordinate is monotone along the ray):
 *   entered(k): every axis has reached the brick's slab      (false ... false true ... true)
 *   left(k):    some axis has gone past the brick's slab     (false ... false true ... true)
 * Sample k belongs to the brick iff entered(k) && !left(k). */
__device__ __forceinline__ void owner_flags(const RaySetup& r, const VrGrid& g, double step, const int bc[3], int k,
                                            bool& entered, bool& left) {
    double s, w;
    sample_sw(r, step, k, s, w);
    entered = true;
    left = false;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        const int c = owner_axis(r, g, s, a);
        if (r.d[a] > 0.0) {
            entered = entered && (c >= bc[a]);
            left = left || (c > bc[a]);
        } else if (r.d[a] < 0.0) {
            entered = entered && (c <= bc[a]);
            left = left || (c < bc[a]);
        } else {
            entered = entered && (c == bc[a]);
        }
    }
}

template <bool WANT_LEFT>
__device__ __forceinline__ bool owner_pred(const RaySetup& r, const VrGrid& g, double step, const int bc[3], int k) {
    bool e, l;
    owner_flags(r, g, step, bc, k, e, l);
    return WANT_LEFT ? l : e;
}

/* Smallest k in [0,K] with pred(k) (pred(K) taken as true); `est` is a guess. */
template <bool WANT_LEFT>
__device__ __forceinline__ int first_true(const RaySetup& r, const VrGrid& g, double step, const int bc[3], int est) {
    const int K = r.K;
    est = est < 0 ? 0 : (est > K ? K : est);
    const bool at = (est == K) || owner_pred<WANT_LEFT>(r, g, step, bc, est);
    const bool before = (est > 0) && owner_pred<WANT_LEFT>(r, g, step, bc, est - 1);
    if (at && !before) return est;
    int lo, hi; /* invariant: pred(lo-1) false (or lo == 0), pred(hi) true */
    if (at) {
        lo = 0;
        hi = est - 1;
    } else {
        lo = est + 1;
        hi = K;
    }
    while (lo < hi) {
        const int mid = lo + ((hi - lo) >> 1);
        if (owner_pred<WANT_LEFT>(r, g, step, bc, mid)) hi = mid;
        else lo = mid + 1;
    }
    return lo;
}

/* The integer sample range [k_lo, k_hi) of the ray that brick bc owns (R6). */
__device__ __forceinline__ void brick_range(const RaySetup& r, const VrGrid& g, double step, const int bc[3],
                                            const int lo[3], const int hi[3], int& k_lo, int& k_hi) {
    k_lo = 0;
    k_hi = 0;
    if (r.K <= 0) return;
    /* approximate clip of the ray against the brick's box: guesses only, and a conservative
     * early out for rays of the rectangle that miss the brick */
    double tin = r.t0, tout = r.t1;
    bool miss = false;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        const bool first = bc[a] == 0, last = bc[a] == g.g[a] - 1;
        if (r.d[a] == 0.0) {
            if ((!first && r.o[a] < (double)lo[a] - 1e-6) || (!last && r.o[a] > (double)hi[a] + 1e-6)) miss = true;
        } else {
            const double inv = 1.0 / r.d[a];
            double ta = ((double)lo[a] - r.o[a]) * inv, tb = ((double)hi[a] - r.o[a]) * inv;
            const bool swap = ta > tb;
            if (swap) {
                const double t = ta;
                ta = tb;
                tb = t;
            }
            /* the outermost bricks own everything beyond the volume's faces (clamped owner) */
            const bool open_in = swap ? last : first, open_out = swap ? first : last;
            if (!open_in && ta > tin) tin = ta;
            if (!open_out && tb < tout) tout = tb;
        }
    }
    if (miss || tout < tin - 1e-6 * (1.0 + fabs(tin))) return;
    const double inv_step = 1.0 / step;
    const double e_lo = ceil((tin - r.t0) * inv_step - 0.5);
    const double e_hi = ceil((tout - r.t0) * inv_step - 0.5);
    const int est_lo = e_lo < 0.0 ? 0 : (e_lo > (double)r.K ? r.K : (int)e_lo);
    const int est_hi = e_hi < 0.0 ? 0 : (e_hi > (double)r.K ? r.K : (int)e_hi);
    k_lo = first_true<false>(r, g, step, bc, est_lo);
    if (k_lo >= r.K) {
        k_hi = k_lo;
        return;
    }
    k_hi = first_true<true>(r, g, step, bc, est_hi);
    if (k_hi < k_lo) k_hi = k_lo;
}

/* ------------------------------------------------------------------------------------------ */
struct Lattice {
    long long q[3]; /* 32.32 fixed point: padded-brick cell coordinate of the sample minus 1/2 */
};

__device__ __forceinline__ long long to_fixed(double x) { return __double2ll_rn(x * 4294967296.0); }

/* Tri-linear interpolation (R3) at a fixed-point brick-local position. PT > 0: the padded
 * edge is a compile-time constant so the 8 loads share one address register pair. */
/* Instrumented variant only: mark brick-store cell `cell` in the touched-cells bitmap. */
__device__ __forceinline__ void mark_cell(unsigned* __restrict__ bitmap, long long cell) {
    atomicOr(bitmap + (cell >> 5), 1u << (unsigned)(cell & 31));
}

/* Brick layouts the kernel is instantiated for:
 *   LAY_LINEAR  x-linear rows of PT (compile time) or g.P cells;
 *   LAY_TILE442 4x4x2-cell micro-tiles, tiles x fastest: per axis two integer operations,
 *               ox(i) = i + (i>>2)*28, oy(j) = 4j + (j>>2)*(SY-16), oz(k) = 16k + (k>>1)*(SZ-32);
 *   LAY_GENERIC any separable layout of VrAxisLayout (micro-tile shape, macro blocks). */
enum { LAY_LINEAR = 0, LAY_TILE442 = 1, LAY_GENERIC = 2 };

template <int LAY>
__device__ __forceinline__ int axis_off(const VrGrid& g, int a, int i) {
    if (LAY == LAY_TILE442) {
        if (a == 0) return i + (i >> 2) * 28;
        if (a == 1) return 4 * i + (i >> 2) * ((int)g.ax[1].hi_stride - 16);
        return 16 * i + (i >> 1) * ((int)g.ax[2].hi_stride - 32);
    }
    return (int)vr_axis_offset(g.ax[a], i);
}

/* The 8 voxels around a lattice position (cell = integer words of L), x fastest in c[]. */
struct Corners {
    float c000, c001, c010, c011, c100, c101, c110, c111;
};

template <int LAY, int PT, bool CLAMP, bool COUNT>
__device__ __forceinline__ void fetch8(const float* __restrict__ brick, const VrGrid& g, const int ext[3], const Lattice& L,
                                       unsigned* __restrict__ bitmap, long long brick_cell0, Corners& C) {
    const int Pe = PT > 0 ? PT : g.P;
    int ix = (int)(L.q[0] >> 32), iy = (int)(L.q[1] >> 32), iz = (int)(L.q[2] >> 32);
    float c000, c001, c010, c011, c100, c101, c110, c111;
    if (LAY == LAY_TILE442 && !CLAMP) {
        /* ghost >= 1: every index is >= 0, so the offsets are
         * unsigned 32-bit and each address is one 32x32+64 multiply-add on a kept base */
        const unsigned ux0 = (unsigned)ix, ux1 = ux0 + 1u, uy0 = (unsigned)iy, uy1 = uy0 + 1u, uz0 = (unsigned)iz, uz1 = uz0 + 1u;
        const unsigned sy = g.ax[1].hi_stride - 16u, sz = g.ax[2].hi_stride - 32u;
        const unsigned ox0 = ux0 + (ux0 >> 2) * 28u, ox1 = ux1 + (ux1 >> 2) * 28u;
        const unsigned oy0 = (uy0 << 2) + (uy0 >> 2) * sy, oy1 = (uy1 << 2) + (uy1 >> 2) * sy;
        const unsigned oz0 = (uz0 << 4) + (uz0 >> 1) * sz, oz1 = (uz1 << 4) + (uz1 >> 1) * sz;
        const unsigned r00 = oz0 + oy0, r01 = oz0 + oy1, r10 = oz1 + oy0, r11 = oz1 + oy1;
        c000 = __ldg(brick + (r00 + ox0));
        c001 = __ldg(brick + (r00 + ox1));
        c010 = __ldg(brick + (r01 + ox0));
        c011 = __ldg(brick + (r01 + ox1));
        c100 = __ldg(brick + (r10 + ox0));
        c101 = __ldg(brick + (r10 + ox1));
        c110 = __ldg(brick + (r11 + ox0));
        c111 = __ldg(brick + (r11 + ox1));
        if (COUNT && bitmap) {
            const long long c0 = brick_cell0 + ox0, c1 = brick_cell0 + ox1;
            mark_cell(bitmap, c0 + r00);
            mark_cell(bitmap, c1 + r00);
            mark_cell(bitmap, c0 + r01);
            mark_cell(bitmap, c1 + r01);
            mark_cell(bitmap, c0 + r10);
            mark_cell(bitmap, c1 + r10);
            mark_cell(bitmap, c0 + r11);
            mark_cell(bitmap, c1 + r11);
        }
    } else if (LAY != LAY_LINEAR) {
        int x0 = ix, x1 = ix + 1, y0 = iy, y1 = iy + 1, z0 = iz, z1 = iz + 1;
        if (CLAMP) { /* ghost = 0: indices leaving the brick's own cells are clamped into them (seams) */
            x0 = min(max(x0, 0), ext[0] - 1), x1 = min(max(x1, 0), ext[0] - 1);
            y0 = min(max(y0, 0), ext[1] - 1), y1 = min(max(y1, 0), ext[1] - 1);
            z0 = min(max(z0, 0), ext[2] - 1), z1 = min(max(z1, 0), ext[2] - 1);
        }
        const int ox0 = axis_off<LAY>(g, 0, x0), ox1 = axis_off<LAY>(g, 0, x1);
        const int oy0 = axis_off<LAY>(g, 1, y0), oy1 = axis_off<LAY>(g, 1, y1);
        const int oz0 = axis_off<LAY>(g, 2, z0), oz1 = axis_off<LAY>(g, 2, z1);
        const int r00 = oz0 + oy0, r01 = oz0 + oy1, r10 = oz1 + oy0, r11 = oz1 + oy1;
        c000 = __ldg(brick + (r00 + ox0));
        c001 = __ldg(brick + (r00 + ox1));
        c010 = __ldg(brick + (r01 + ox0));
        c011 = __ldg(brick + (r01 + ox1));
        c100 = __ldg(brick + (r10 + ox0));
        c101 = __ldg(brick + (r10 + ox1));
        c110 = __ldg(brick + (r11 + ox0));
        c111 = __ldg(brick + (r11 + ox1));
        if (COUNT && bitmap) {
            mark_cell(bitmap, brick_cell0 + (r00 + ox0));
            mark_cell(bitmap, brick_cell0 + (r00 + ox1));
            mark_cell(bitmap, brick_cell0 + (r01 + ox0));
            mark_cell(bitmap, brick_cell0 + (r01 + ox1));
            mark_cell(bitmap, brick_cell0 + (r10 + ox0));
            mark_cell(bitmap, brick_cell0 + (r10 + ox1));
            mark_cell(bitmap, brick_cell0 + (r11 + ox0));
            mark_cell(bitmap, brick_cell0 + (r11 + ox1));
        }
    } else if (!CLAMP) {
        const float* p = brick + ((long long)(iz * Pe + iy) * Pe + ix);
        c000 = __ldg(p);
        c001 = __ldg(p + 1);
        c010 = __ldg(p + Pe);
        c011 = __ldg(p + Pe + 1);
        c100 = __ldg(p + Pe * Pe);
        c101 = __ldg(p + Pe * Pe + 1);
        c110 = __ldg(p + Pe * Pe + Pe);
        c111 = __ldg(p + Pe * Pe + Pe + 1);
        if (COUNT && bitmap) {
            const long long c = brick_cell0 + (p - brick);
            mark_cell(bitmap, c);
            mark_cell(bitmap, c + 1);
            mark_cell(bitmap, c + Pe);
            mark_cell(bitmap, c + Pe + 1);
            mark_cell(bitmap, c + Pe * Pe);
            mark_cell(bitmap, c + Pe * Pe + 1);
            mark_cell(bitmap, c + Pe * Pe + Pe);
            mark_cell(bitmap, c + Pe * Pe + Pe + 1);
        }
    } else {
        /* ghost = 0: indices leaving the brick's own cells are clamped into them (seams) */
        const int x0 = min(max(ix, 0), ext[0] - 1), x1 = min(max(ix + 1, 0), ext[0] - 1);
        const int y0 = min(max(iy, 0), ext[1] - 1), y1 = min(max(iy + 1, 0), ext[1] - 1);
        const int z0 = min(max(iz, 0), ext[2] - 1), z1 = min(max(iz + 1, 0), ext[2] - 1);
        const long long r00 = (long long)(z0 * Pe + y0) * Pe, r01 = (long long)(z0 * Pe + y1) * Pe;
        const long long r10 = (long long)(z1 * Pe + y0) * Pe, r11 = (long long)(z1 * Pe + y1) * Pe;
        c000 = __ldg(brick + r00 + x0);
        c001 = __ldg(brick + r00 + x1);
        c010 = __ldg(brick + r01 + x0);
        c011 = __ldg(brick + r01 + x1);
        c100 = __ldg(brick + r10 + x0);
        c101 = __ldg(brick + r10 + x1);
        c110 = __ldg(brick + r11 + x0);
        c111 = __ldg(brick + r11 + x1);
        if (COUNT && bitmap) {
            mark_cell(bitmap, brick_cell0 + r00 + x0);
            mark_cell(bitmap, brick_cell0 + r00 + x1);
            mark_cell(bitmap, brick_cell0 + r01 + x0);
            mark_cell(bitmap, brick_cell0 + r01 + x1);
            mark_cell(bitmap, brick_cell0 + r10 + x0);
            mark_cell(bitmap, brick_cell0 + r10 + x1);
            mark_cell(bitmap, brick_cell0 + r11 + x0);
            mark_cell(bitmap, brick_cell0 + r11 + x1);
        }
    }
    C.c000 = c000, C.c001 = c001, C.c010 = c010, C.c011 = c011;
    C.c100 = c100, C.c101 = c101, C.c110 = c110, C.c111 = c111;
}

/* Tri-linear interpolation (R3): the fraction words of L are the float32 weights. */
__device__ __forceinline__ float lerp8(const Corners& C, const Lattice& L) {
    const float fx = __uint_as_float(0x3F800000u | ((unsigned)L.q[0] >> 9)) - 1.0f;
    const float fy = __uint_as_float(0x3F800000u | ((unsigned)L.q[1] >> 9)) - 1.0f;
    const float fz = __uint_as_float(0x3F800000u | ((unsigned)L.q[2] >> 9)) - 1.0f;
    const float c00 = fmaf(fx, C.c001 - C.c000, C.c000);
    const float c01 = fmaf(fx, C.c011 - C.c010, C.c010);
    const float c10 = fmaf(fx, C.c101 - C.c100, C.c100);
    const float c11 = fmaf(fx, C.c111 - C.c110, C.c110);
    const float c0 = fmaf(fy, c01 - c00, c00);
    const float c1 = fmaf(fy, c11 - c10, c10);
    return fmaf(fz, c1 - c0, c0);
}

template <int LAY, int PT, bool CLAMP, bool COUNT>
__device__ __forceinline__ float trilinear(const float* __restrict__ brick, const VrGrid& g, const int ext[3], const Lattice& L,
                                           unsigned* __restrict__ bitmap, long long brick_cell0) {
    Corners C;
    fetch8<LAY, PT, CLAMP, COUNT>(brick, g, ext, L, bitmap, brick_cell0, C);
    return lerp8(C, L);
}

struct Accum {
    float r, g, b, a; /* ALPHA: premultiplied colour and opacity; MIP: r = running max */
};

/* The LUT as the kernel sees it: (entry, delta) pairs interleaved in shared memory, addressed
 * through one 32-bit shared-window address kept in a register. */
struct LutView {
    unsigned base; /* shared-memory byte address of pair 0 */
};

template <int OFF>
__device__ __forceinline__ float4 lds128(unsigned addr) {
    float4 v;
    asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4+%5];"
                 : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w)
                 : "r"(addr), "n"(OFF));
    return v;
}
__device__ __forceinline__ float lg2_approx(float x) {
    float y;
    asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ float ex2_approx(float x) {
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

/* R7: classification and opacity of a sample standing for a path of length w; R8 blending.
 * alpha = 1 - (1-a)^w = 1 - 2^(w log2(1-a)) on the two MUFU approximations (2^-22 relative,
 * DESIGN.md "Tolerances"); a = 1 gives log2(0) = -inf and alpha = 1, a = 0 gives alpha = 0. */
__device__ __forceinline__ void shade_alpha(Accum& acc, float v, float w, const LutView& lut, const VrLut& P) {
    const float u = __saturatef((v - P.vmin) * P.inv_range);
    const float x = u * P.scale;
    const int i = min((int)x, P.nm2);
    const float f = x - (float)i;
    const unsigned a = lut.base + 32u * (unsigned)i;
    const float4 e = lds128<0>(a), dl = lds128<16>(a);
    const float cr = fmaf(f, dl.x, e.x), cg = fmaf(f, dl.y, e.y), cb = fmaf(f, dl.z, e.z), ca = fmaf(f, dl.w, e.w);
    const float alpha = 1.0f - ex2_approx(w * lg2_approx(1.0f - ca));
    const float ta = (1.0f - acc.a) * alpha;
    acc.r = fmaf(ta, cr, acc.r);
    acc.g = fmaf(ta, cg, acc.g);
    acc.b = fmaf(ta, cb, acc.b);
    acc.a += ta;
}

template <int MODE, int LAY, int PT, bool CLAMP, bool COUNT>
__global__ void __launch_bounds__(VR_RAYCAST_THREADS, VR_MIN_CTAS)
vr_raycast_kernel(const VrRaycastParams prm) {
    /* dynamic: 2 * lut.n float4 (ALPHA) - a 256-entry table takes 8 KB, not the 32 KB of the
     * largest one, and what it does not take stays L1 cache */
    extern __shared__ float4 s_lut[];
    __shared__ double s_minv[16];

    const VrGrid& g = prm.grid;
    const int lane = threadIdx.x & 31;
    if (MODE == VR_ALPHA) {
        for (int i = threadIdx.x; i < prm.lut.n; i += blockDim.x) {
            s_lut[2 * i] = prm.lut.base[i];
            s_lut[2 * i + 1] = prm.lut.delta[i];
        }
    }
    if (threadIdx.x < 16) s_minv[threadIdx.x] = prm.vs->Minv[threadIdx.x];
    __syncthreads();
    if (prm.vs->singular) return;

    const int W = prm.vs->W, H = prm.vs->H;
    const int total = prm.vs->total_items;
    const double step = prm.step;
    const float tau = prm.tau;
    LutView lut;
    lut.base = 0;
    if (MODE == VR_ALPHA) {
        lut.base = (unsigned)__cvta_generic_to_shared(s_lut);
        asm volatile("" : "+r"(lut.base)); /* one register, not rebuilt per sample */
    }
    /* MIP may stop where the output saturates (vmax) or at the global maximum of the data when
     * it is known ("the maximum pixel value (defined by the global maximum of the data)") */
    const float mip_stop = fminf(prm.lut.vmax, prm.vs->data_max);
    unsigned long long nsamples = 0;

    /* one atomic per item; the next item is requested before the current one is processed */
    unsigned next = 0;
    if (lane == 0) next = atomicAdd(&prm.vs_rw->work_counter, 1u);
    next = __shfl_sync(FULL_MASK, next, 0);

    while (next < (unsigned)total) {
        const int item = (int)next;
        if (lane == 0) next = atomicAdd(&prm.vs_rw->work_counter, 1u);

        /* item -> (order position, tile) by binary search in the exclusive prefix */
        int lo_q = 0, hi_q = g.nbricks - 1;
        while (lo_q < hi_q) {
            const int mid = (lo_q + hi_q + 1) >> 1;
            if (__ldg(prm.item_prefix + mid) <= item) lo_q = mid;
            else hi_q = mid - 1;
        }
        const int b = __ldg(prm.order + lo_q);
        const int local = item - __ldg(prm.item_prefix + lo_q);
        const VrBrickView bvw = prm.bv[b];
        const int ty = local / bvw.tiles_x, tx = local - ty * bvw.tiles_x;
        const int pi = bvw.lx0 + tx * VR_TILE_W + (lane & 7);
        const int pj = bvw.ly0 + ty * VR_TILE_H + (lane >> 3);
        const bool in_launch = pi < bvw.lx1 && pj < bvw.ly1;
        const bool in_rect = in_launch && pi >= bvw.rx0 && pi < bvw.rx1 && pj >= bvw.ry0 && pj < bvw.ry1;

        int bc[3], blo[3], bhi[3], ext[3];
        vr_brick_coords(g, b, bc);
        vr_brick_core(g, bc, blo, bhi);
#pragma unroll
        for (int a = 0; a < 3; ++a) ext[a] = bhi[a] - blo[a] + 2 * g.ghost;
        const float* __restrict__ brick = prm.bricks + (long long)b * g.slot;
        asm volatile("" : "+l"(brick)); /* keep the base in registers: do not rebuild it per load */

        RaySetup ray;
        ray.K = 0;
        int k_lo = 0, k_hi = 0;
        if (in_rect) {
            ray_setup(s_minv, W, H, pi, pj, g, step, ray);
            brick_range(ray, g, step, bc, blo, bhi, k_lo, k_hi);
        }
        /* lattice samples: k in [k_lo, k_lat); samples k >= K-2 (whose interval may be clipped
         * by the exit point) are evaluated one by one in FP64 below */
        const int k_lat = min(k_hi, max(k_lo, ray.K - 2));
        int n = k_lat - k_lo;

        Accum acc;
        acc.r = (MODE == VR_MIP) ? -INFINITY : 0.0f;
        acc.g = acc.b = acc.a = 0.0f;
        Lattice L;
        long long D[3];
        if (n > 0) {
            double s, w;
            sample_sw(ray, step, k_lo, s, w);
#pragma unroll
            for (int a = 0; a < 3; ++a) {
                const double p = VR_FMA(s, ray.d[a], ray.o[a]);
                L.q[a] = to_fixed(p - ((double)(blo[a] - g.ghost) + 0.5));
                D[a] = to_fixed(step * ray.d[a]);
            }
        } else {
            L.q[0] = L.q[1] = L.q[2] = 0;
            D[0] = D[1] = D[2] = 0;
        }
        bool stopped = (MODE == VR_ALPHA) ? !(acc.a < tau) : false;
        bool active = n > 0 && !stopped;
        /* With step < 1 consecutive samples of a ray often fall into the same cell: the 8
         * voxels stay in registers and only the weights change (fewer L1 wavefronts, the
         * bound of densely sampled views). */
        Corners C;
        int pcx = INT_MIN, pcy = 0, pcz = 0;
        while (__any_sync(FULL_MASK, active)) {
            if (active) {
                const int cx = (int)(L.q[0] >> 32), cy = (int)(L.q[1] >> 32), cz = (int)(L.q[2] >> 32);
                if (!VR_REUSE || cx != pcx || cy != pcy || cz != pcz) {
                    fetch8<LAY, PT, CLAMP, COUNT>(brick, g, ext, L, prm.bitmap, (long long)b * g.slot, C);
                    pcx = cx, pcy = cy, pcz = cz;
                }
                const float v = lerp8(C, L);
                if (COUNT) ++nsamples;
                if (MODE == VR_MIP) {
                    acc.r = fmaxf(acc.r, v);
                    stopped = acc.r >= mip_stop;
                } else {
                    shade_alpha(acc, v, prm.stepf, lut, prm.lut);
                    stopped = !(acc.a < tau);
                }
                L.q[0] += D[0], L.q[1] += D[1], L.q[2] += D[2];
                --n;
                active = n > 0 && !stopped;
            }
        }
        /* the (at most two) samples next to the exit point */
        const int k_tail = max(k_lat, k_lo);
        if (__any_sync(FULL_MASK, k_tail < k_hi && !stopped)) {
#if VR_RECOMPUTE_TAIL
            if (k_tail < k_hi && !stopped) {
                int qi = pi, qj = pj; /* opaque copies: the ray is rebuilt, not kept in registers */
                asm volatile("" : "+r"(qi), "+r"(qj));
                ray_setup(s_minv, W, H, qi, qj, g, step, ray);
            }
#endif
            for (int k = k_tail; k < k_hi && !stopped; ++k) {
                double s, w;
                if (!sample_sw(ray, step, k, s, w)) continue;
#pragma unroll
                for (int a = 0; a < 3; ++a) {
                    const double p = VR_FMA(s, ray.d[a], ray.o[a]);
                    L.q[a] = to_fixed(p - ((double)(blo[a] - g.ghost) + 0.5));
                }
                const float v = trilinear<LAY, PT, CLAMP, COUNT>(brick, g, ext, L, prm.bitmap, (long long)b * g.slot);
                if (COUNT) ++nsamples;
                if (MODE == VR_MIP) {
                    acc.r = fmaxf(acc.r, v);
                    stopped = acc.r >= mip_stop;
                } else {
                    shade_alpha(acc, v, (float)w, lut, prm.lut);
                    stopped = !(acc.a < tau);
                }
            }
        }

        /* row a8: one sub-image pixel per pixel of the launch rectangle */
        if (in_launch) {
            const long long off = bvw.sub_offset + (long long)(pj - bvw.ly0) * (bvw.lx1 - bvw.lx0) + (pi - bvw.lx0);
            if (MODE == VR_ALPHA) reinterpret_cast<float4*>(prm.sub)[off] = make_float4(acc.r, acc.g, acc.b, acc.a);
            else reinterpret_cast<float*>(prm.sub)[off] = acc.r;
        }
        next = __shfl_sync(FULL_MASK, next, 0);
    }
    if (COUNT) {
        for (int o = 16; o > 0; o >>= 1) nsamples += __shfl_xor_sync(FULL_MASK, nsamples, o);
        if (lane == 0 && nsamples) atomicAdd(&prm.vs_rw->samples, nsamples);
    }
}

/* ------------------------------------------------------------------------------------------ */
/* Persistent grid: resident CTAs per SM (for this instance and its shared memory) x SMs,
 * but no more CTAs than there are groups of 8 work items. */
template <int MODE, int LAY, int PT, bool CLAMP, bool COUNT>
static cudaError_t launch_variant(const VrRaycastParams& p, long long items, cudaStream_t st) {
    static int sms = 0, cached_per_sm = 0;
    static size_t cached_smem = (size_t)-1;
    const size_t smem = MODE == VR_ALPHA ? 2 * sizeof(float4) * (size_t)p.lut.n : 0;
    if (smem != cached_smem) {
        int dev = 0;
        cudaError_t e = cudaGetDevice(&dev);
        if (e == cudaSuccess) e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        if (e == cudaSuccess)
            e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&cached_per_sm, vr_raycast_kernel<MODE, LAY, PT, CLAMP, COUNT>,
                                                              VR_RAYCAST_THREADS, smem);
        if (e != cudaSuccess) return e;
        if (cached_per_sm < 1) return cudaErrorLaunchOutOfResources;
        cached_smem = smem;
    }
    long long ctas = (long long)sms * cached_per_sm;
    const long long want = (items + (VR_RAYCAST_THREADS / 32) - 1) / (VR_RAYCAST_THREADS / 32);
    if (ctas > want) ctas = want < 1 ? 1 : want;
    vr_raycast_kernel<MODE, LAY, PT, CLAMP, COUNT><<<(int)ctas, VR_RAYCAST_THREADS, smem, st>>>(p);
    return cudaGetLastError();
}

static bool is_tile442(const VrGrid& g) {
    return g.layout == VR_LAYOUT_TILED && g.tl[0] == 2 && g.tl[1] == 2 && g.tl[2] == 1 && g.ml[0] == 0 && g.ml[1] == 0 &&
           g.ml[2] == 0;
}

template <int MODE, bool COUNT>
static cudaError_t launch_mode(const VrRaycastParams& p, long long ctas, cudaStream_t st) {
    const bool clamp = p.grid.ghost == 0;
    if (p.grid.layout == VR_LAYOUT_LINEAR) {
        if (clamp) return launch_variant<MODE, LAY_LINEAR, 0, true, COUNT>(p, ctas, st);
        switch (p.grid.P) {
            case 258: return launch_variant<MODE, LAY_LINEAR, 258, false, COUNT>(p, ctas, st);
            case 514: return launch_variant<MODE, LAY_LINEAR, 514, false, COUNT>(p, ctas, st);
            default: return launch_variant<MODE, LAY_LINEAR, 0, false, COUNT>(p, ctas, st);
        }
    }
    if (is_tile442(p.grid))
        return clamp ? launch_variant<MODE, LAY_TILE442, 0, true, COUNT>(p, ctas, st)
                     : launch_variant<MODE, LAY_TILE442, 0, false, COUNT>(p, ctas, st);
    return clamp ? launch_variant<MODE, LAY_GENERIC, 0, true, COUNT>(p, ctas, st)
                 : launch_variant<MODE, LAY_GENERIC, 0, false, COUNT>(p, ctas, st);
}

cudaError_t vr_launch_raycast(const VrRaycastParams& p, long long ctas, bool count, cudaStream_t st) {
    if (p.mode == VR_ALPHA) return count ? launch_mode<VR_ALPHA, true>(p, ctas, st) : launch_mode<VR_ALPHA, false>(p, ctas, st);
    return count ? launch_mode<VR_MIP, true>(p, ctas, st) : launch_mode<VR_MIP, false>(p, ctas, st);
}
