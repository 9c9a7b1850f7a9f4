/*
 * vr_march.cuh -- device helpers shared by the two ray-marching kernels (vr_raycast.cu: one
 * brick per ray segment and sub-image, sort-last; vr_fused.cu: one ray through all bricks):
 * FP64 ray set-up and the exact integer sample range a brick owns (R1, R2, R4, R5, R6), the
 * 32.32 fixed-point lattice, the 8-voxel fetch for each brick layout, float32 tri-linear
 * interpolation (R3) and classification / blending (R7, R8).
 */
#ifndef VR_MARCH_CUH
#define VR_MARCH_CUH

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
    double step; /* sample spacing along this ray (R5); per ray when the caller asks for the paper's rule (R18) */
    int K; /* number of scheduled samples; 0 = miss */
    double inv_d[3], inv_step; /* 1/d_a (0 where d_a == 0) and 1/step: for the estimates of brick_range only */
};

/* R1, R2: pixel (i,j), centres at half-integers, row 0 at the bottom; ray from the near plane
 * (clip z = -1) to the far plane (+1). R4: slab test against the closed global box.
 * step > 0: the caller's spacing; step == 0: R18, the paper's "at least one sample for each voxel
 * intersected", one sample per unit advance along the major axis, 1 / max|d_a|. */
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
    if (step == 0.0) {
        double m = fabs(r.d[0]);
        if (fabs(r.d[1]) > m) m = fabs(r.d[1]);
        if (fabs(r.d[2]) > m) m = fabs(r.d[2]);
        step = VR_DIV(1.0, m);
    }
    r.step = step;

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
#pragma unroll
    for (int a = 0; a < 3; ++a) r.inv_d[a] = r.d[a] == 0.0 ? 0.0 : 1.0 / r.d[a];
    r.inv_step = 1.0 / step;
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

/* The ray of pixel p = j*W + i from the frame's ray table (VrRaycastParams::rays, layout in vr_internal.cuh): the values
 * ray_setup computed, bit for bit. FULL also fills the reciprocals brick_range's ESTIMATES use, from float32
 * reciprocals (relative error 1e-7: < 1e-3 voxel on the longest ray, a tenth of the margin of brick_range's early
 * out; a wrong guess only costs a bisection). step_fixed > 0: the caller's spacing (not stored); 0: per ray (R18). */
/* the int plane (K) and, 16-byte aligned behind it, the double plane (per-ray step) */
__device__ __forceinline__ const int* ray_k_plane(const double2* rays, long long plane) { return reinterpret_cast<const int*>(rays + 4 * plane); }
__device__ __forceinline__ const double* ray_step_plane(const double2* rays, long long plane) {
    return reinterpret_cast<const double*>(reinterpret_cast<const char*>(rays + 4 * plane) + ((plane * 4 + 15) & ~15ll));
}

template <bool FULL>
__device__ __forceinline__ void ray_load(const double2* __restrict__ rays, long long plane, long long p, double step_fixed, RaySetup& r) {
    const double2 a0 = __ldg(rays + p), a1 = __ldg(rays + plane + p), a2 = __ldg(rays + 2 * plane + p), a3 = __ldg(rays + 3 * plane + p);
    r.K = __ldg(ray_k_plane(rays, plane) + p);
    r.o[0] = a0.x, r.o[1] = a0.y, r.o[2] = a1.x;
    r.d[0] = a1.y, r.d[1] = a2.x, r.d[2] = a2.y;
    r.t0 = a3.x, r.t1 = a3.y;
    r.step = step_fixed > 0.0 ? step_fixed : __ldg(ray_step_plane(rays, plane) + p);
    if (FULL) {
#pragma unroll
        for (int a = 0; a < 3; ++a) r.inv_d[a] = r.d[a] == 0.0 ? 0.0 : (double)__frcp_rn((float)r.d[a]);
        r.inv_step = (double)__frcp_rn((float)r.step);
    }
}

__device__ __forceinline__ void ray_store(double2* __restrict__ rays, long long plane, long long p, bool step_fixed, const RaySetup& r) {
    rays[p] = make_double2(r.o[0], r.o[1]);
    rays[plane + p] = make_double2(r.o[2], r.d[0]);
    rays[2 * plane + p] = make_double2(r.d[1], r.d[2]);
    rays[3 * plane + p] = make_double2(r.t0, r.t1);
    const_cast<int*>(ray_k_plane(rays, plane))[p] = r.K;
    if (!step_fixed) const_cast<double*>(ray_step_plane(rays, plane))[p] = r.step;
}

/* R5: sample k stands for the interval [t0 + k step, min(t0 + (k+1) step, t1)]: s = its
 * midpoint, w = its length; intervals of non-positive length are dropped. */
__device__ __forceinline__ bool sample_sw(const RaySetup& r, int k, double& s, double& w) {
    const double step = r.step;
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
__device__ __forceinline__ void owner_flags(const RaySetup& r, const VrGrid& g, const int bc[3], int k,
                                            bool& entered, bool& left) {
    double s, w;
    sample_sw(r, k, s, w);
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
__device__ __forceinline__ bool owner_pred(const RaySetup& r, const VrGrid& g, const int bc[3], int k) {
    bool e, l;
    owner_flags(r, g, bc, k, e, l);
    return WANT_LEFT ? l : e;
}

/* Smallest k in [0,K] with pred(k) (pred(K) taken as true); `est` is a guess. */
template <bool WANT_LEFT>
__device__ __forceinline__ int first_true(const RaySetup& r, const VrGrid& g, const int bc[3], int est) {
    const int K = r.K;
    est = est < 0 ? 0 : (est > K ? K : est);
    const bool at = (est == K) || owner_pred<WANT_LEFT>(r, g, bc, est);
    const bool before = (est > 0) && owner_pred<WANT_LEFT>(r, g, bc, est - 1);
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
        if (owner_pred<WANT_LEFT>(r, g, bc, mid)) hi = mid;
        else lo = mid + 1;
    }
    return lo;
}

/* The integer sample range [k_lo, k_hi) of the ray that brick bc owns (R6). */
__device__ __forceinline__ void brick_range(const RaySetup& r, const VrGrid& g, const int bc[3],
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
            const double inv = r.inv_d[a];
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
    const double inv_step = r.inv_step;
    const double e_lo = ceil((tin - r.t0) * inv_step - 0.5);
    const double e_hi = ceil((tout - r.t0) * inv_step - 0.5);
    const int est_lo = e_lo < 0.0 ? 0 : (e_lo > (double)r.K ? r.K : (int)e_lo);
    const int est_hi = e_hi < 0.0 ? 0 : (e_hi > (double)r.K ? r.K : (int)e_hi);
    k_lo = first_true<false>(r, g, bc, est_lo);
    if (k_lo >= r.K) {
        k_hi = k_lo;
        return;
    }
    k_hi = first_true<true>(r, g, bc, est_hi);
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

/* The voxel load of the 4x4x2 path. VR_LDG_L2_64B (build-time experiment, profiles/r2_c3_experiments.md): the L2::64B
 * prefetch-size hint halves the DRAM bytes of a miss (probe: 63.8 instead of 127.3 bytes per load) but not the rate at
 * which misses are served, and the second half of a micro-tile then costs a request of its own. */
__device__ __forceinline__ float vr_ldg(const float* p) {
#ifdef VR_LDG_L2_64B
    float v;
    asm volatile("ld.global.nc.L1::no_allocate.L2::64B.f32 %0, [%1];" : "=f"(v) : "l"(p));
    return v;
#elif defined(VR_LDG_L2_64B_ALLOC)
    float v;
    asm volatile("ld.global.nc.L2::64B.f32 %0, [%1];" : "=f"(v) : "l"(p));
    return v;
#else
    return __ldg(p);
#endif
}

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
        c000 = vr_ldg(brick + (r00 + ox0));
        c001 = vr_ldg(brick + (r00 + ox1));
        c010 = vr_ldg(brick + (r01 + ox0));
        c011 = vr_ldg(brick + (r01 + ox1));
        c100 = vr_ldg(brick + (r10 + ox0));
        c101 = vr_ldg(brick + (r10 + ox1));
        c110 = vr_ldg(brick + (r11 + ox0));
        c111 = vr_ldg(brick + (r11 + ox1));
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

/* R14, the rare path: lerp8 gave NaN, i.e. some of the 8 voxels are blanked. N = tri-linear weight on the
 * NaN corners; N > 4e-6: the sample is dropped (NaN stays); otherwise the NaN corners are left out and the
 * others renormalised - continuous where a sample sits on a cell boundary next to a blanked voxel. */
static __device__ __forceinline__ float lerp8_blanked_values(float c0, float c1, float c2, float c3, float c4, float c5, float c6,
                                                         float c7, float fx, float fy, float fz) {
    const float c[8] = {c0, c1, c2, c3, c4, c5, c6, c7};
    float N = 0.0f, acc = 0.0f;
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        const float w = ((i & 1) ? fx : 1.0f - fx) * ((i & 2) ? fy : 1.0f - fy) * ((i & 4) ? fz : 1.0f - fz);
        if (c[i] != c[i]) N += w;
        else acc = fmaf(w, c[i], acc);
    }
    return N > 4e-6f ? __int_as_float(0x7fc00000) : acc / (1.0f - N);
}
/* everything by value, in registers: a by-reference call would keep the lattice and the voxels in local memory */
__device__ __forceinline__ float lerp8_blanked(const Corners& C, const Lattice& L) {
    const float fx = __uint_as_float(0x3F800000u | ((unsigned)L.q[0] >> 9)) - 1.0f;
    const float fy = __uint_as_float(0x3F800000u | ((unsigned)L.q[1] >> 9)) - 1.0f;
    const float fz = __uint_as_float(0x3F800000u | ((unsigned)L.q[2] >> 9)) - 1.0f;
    return lerp8_blanked_values(C.c000, C.c001, C.c010, C.c011, C.c100, C.c101, C.c110, C.c111, fx, fy, fz);
}

template <int LAY, int PT, bool CLAMP, bool COUNT>
__device__ __forceinline__ float trilinear(const float* __restrict__ brick, const VrGrid& g, const int ext[3], const Lattice& L,
                                           unsigned* __restrict__ bitmap, long long brick_cell0) {
    Corners C;
    fetch8<LAY, PT, CLAMP, COUNT>(brick, g, ext, L, bitmap, brick_cell0, C);
    float v = lerp8(C, L);
    if (v != v) v = lerp8_blanked(C, L); /* R14 */
    return v;
}

/* R19: how many lattice steps (at least 1, at most n) can be taken from position L without leaving the
 * 8x8x8 macro-cell it is in. An UNDER-estimate by construction (quotients rounded down from values scaled
 * down by 2^-20), so every position stepped over lies inside the macro-cell; landing short only means
 * another leap. 32.32 fixed point: a macro-cell spans 2^35 units per axis. */
__device__ __forceinline__ int leap_steps(const Lattice& L, const long long D[3], int n) {
    float t = (float)n;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        const long long d = D[a];
        if (d != 0) {
            const long long lo = L.q[a] & ~((1ll << 35) - 1);
            /* d > 0: positions j with q + j d < lo + 2^35 are inside: ceil(dist / d) of them; d < 0: floor((q - lo) / -d) + 1 */
            const long long dist = d > 0 ? lo + (1ll << 35) - L.q[a] : L.q[a] - lo;
            const float e = __fdividef(__ll2float_rz(dist), __ll2float_ru(d > 0 ? d : -d)) * 0.999999f;
            t = fminf(t, d > 0 ? e : e + 1.0f);
        }
    }
    const int j = (int)t; /* rounds toward zero */
    return j < 1 ? 1 : j;
}

struct Accum {
    float r, g, b, a; /* ALPHA: premultiplied colour and opacity; MIP: r = running max */
};

/* The LUT as the kernel sees it: (entry, delta) pairs interleaved in shared memory, addressed
 * through one 32-bit shared-window address kept in a register. */
struct LutView {
    unsigned base;   /* shared-memory byte address of pair 0 (replicated layout: of this lane's copy of entry 0) */
    unsigned stride; /* replicated layout: bytes from entry i to entry i + 1 of the same copy */
};

/* Replicated layout (the ray-cast kernel): a 128-bit shared load is served a quarter-warp (8 lanes x 16 bytes = all 32
 * banks) at a time, and the lanes of a quarter read unrelated entries on noisy data: with one table, 8 lanes on 4 (pairs
 * at 32-byte stride) bank groups cost 13.7 wavefronts per load instead of 4 (ncu, c1: 71 % of all shared wavefronts were
 * conflicts). So the table is stored `copies` times, entry i of copy c at (i * copies + c) * 16 bytes, and lane l reads copy
 * l mod copies - its own bank group: no conflicts at copies = 8. Only the entries are stored; the difference to the next
 * entry is the same float32 subtraction the host made for the paired layout. copies = 8 for n <= 256 (32 KB), 4 / 2 above.
 * Sparsely sampled views (the 103 GB cube: every sample misses L2, L1 capacity decides how often a ray finds its previous
 * sample's lines again) keep ONE copy (4 KB): with 32 KB of table per CTA c3 lost 7 % (ramp) to 16 % (translucent). */
__host__ __device__ __forceinline__ int vr_lut_copies(int n, bool sparse) { return sparse ? 1 : (n <= 256 ? 8 : (n <= 512 ? 4 : 2)); }

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
/* classification (the table's interpolated entry for value v) and blending, separately: the texture arm looks at the
 * entry's opacity before it blends (R20's guard). shade_alpha = the two in a row, the same operations as ever. */
template <bool REP = false>
__device__ __forceinline__ float4 classify_alpha(float v, const LutView& lut, const VrLut& P) {
    const float u = __saturatef((v - P.vmin) * P.inv_range);
    const float x = u * P.scale;
    const int i = min((int)x, P.nm2);
    const float f = x - (float)i;
    float4 e, dl;
    if (REP) {
        const unsigned a = lut.base + lut.stride * (unsigned)i;
        e = lds128<0>(a);
        const float4 e1 = lds128<0>(a + lut.stride);
        dl = make_float4(e1.x - e.x, e1.y - e.y, e1.z - e.z, e1.w - e.w);
    } else {
        const unsigned a = lut.base + 32u * (unsigned)i;
        e = lds128<0>(a), dl = lds128<16>(a);
    }
    return make_float4(fmaf(f, dl.x, e.x), fmaf(f, dl.y, e.y), fmaf(f, dl.z, e.z), fmaf(f, dl.w, e.w));
}

__device__ __forceinline__ void blend_alpha(Accum& acc, float v, float w, const float4 c) {
    const float alpha = 1.0f - ex2_approx(w * lg2_approx(1.0f - c.w));
    /* R14: a dropped sample arrives as NaN. It classifies harmlessly (the saturation maps it to entry 0);
     * its opacity is forced to 0. MIP needs nothing: fmaxf ignores NaN. */
    const float ta = (v == v) ? (1.0f - acc.a) * alpha : 0.0f;
    acc.r = fmaf(ta, c.x, acc.r);
    acc.g = fmaf(ta, c.y, acc.g);
    acc.b = fmaf(ta, c.z, acc.b);
    acc.a += ta;
}

template <bool REP = false>
__device__ __forceinline__ void shade_alpha(Accum& acc, float v, float w, const LutView& lut, const VrLut& P) {
    blend_alpha(acc, v, w, classify_alpha<REP>(v, lut, P));
}

#endif
