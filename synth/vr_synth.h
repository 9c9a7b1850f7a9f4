/*
 * vr_synth.h -- seeded synthetic INPUT generator (radio-spectral-cube stand-ins).
 *
 * This module makes inputs only. It holds none of the renderer's arithmetic
 * (no ray, no interpolation, no transfer function, no compositing) and is the
 * one piece of code the CPU oracle (oracle/) and the CUDA path
 * (paper_1205_0282_b200/) are both allowed to see. Recipe: DESIGN.md
 * "Synthetic inputs"; it stands in for the HIPASS/GASS/N-body cubes of the
 * paper's Table 1, which are not available here.
 *
 * The same functions compile for the host (gcc, -ffp-contract=off) and for the
 * device (nvcc, -fmad=false). Every floating-point step is an individually
 * IEEE-rounded operation (+, *, /, sqrt, fma), so host and device produce
 * bit-identical voxels; tests/test_synth.py and tests/test_gpu_parity.py (test_device_generator_is_the_host_generator) check it.
 *
 * voxel(x,y,z) = noise(seed, linear index)                 i.i.d. N(0,1)
 *              + sum over sources s (ascending s) of
 *                peak_s * gx_s[x-x0_s] * gy_s[y-y0_s] * gz_s[z-z0_s]
 *              + ramp * (z + 1/2) / nz                      continuum-like gradient
 * kind VS_NBODY (the paper's other data family, Table 1 "Nbody": a density cube, zero where
 * there are no particles): no noise term, and the sources are extended halos (vr_synth_cpu.c).
 */
#ifndef VR_SYNTH_H
#define VR_SYNTH_H

#include <stdint.h>

#ifdef __CUDACC__
#define VS_HD __host__ __device__ __forceinline__
#else
#define VS_HD static inline
#endif

#if defined(__CUDA_ARCH__)
#define VS_FMUL(a, b) __fmul_rn((a), (b))
#define VS_FADD(a, b) __fadd_rn((a), (b))
#define VS_DMUL(a, b) __dmul_rn((a), (b))
#define VS_DADD(a, b) __dadd_rn((a), (b))
#define VS_DDIV(a, b) __ddiv_rn((a), (b))
#define VS_DSQRT(a) __dsqrt_rn((a))
#define VS_FMA(a, b, c) __fma_rn((a), (b), (c))
#define VS_CLZ64(x) __clzll((long long)(x))
#else
#include <math.h>
#define VS_FMUL(a, b) ((float)((float)(a) * (float)(b)))
#define VS_FADD(a, b) ((float)((float)(a) + (float)(b)))
#define VS_DMUL(a, b) ((double)(a) * (double)(b))
#define VS_DADD(a, b) ((double)(a) + (double)(b))
#define VS_DDIV(a, b) ((double)(a) / (double)(b))
#define VS_DSQRT(a) sqrt((double)(a))
#define VS_FMA(a, b, c) fma((double)(a), (double)(b), (double)(c))
#define VS_CLZ64(x) __builtin_clzll((unsigned long long)(x))
#endif

#define VS_CELL 32 /* edge of the source-lookup cells, voxels */

/* Plain data, host or device pointers depending on where it is used. */
typedef struct vs_cube {
    uint64_t seed;
    int64_t nx, ny, nz;
    double ramp;         /* amplitude of the spectral-axis gradient (0 = none) */
    int32_t nsrc;
    /* per source: integer box origin, box lengths, peak, offsets into prof[] */
    const int32_t* x0; const int32_t* y0; const int32_t* z0;
    const int32_t* lx; const int32_t* ly; const int32_t* lz;
    const float* peak;
    const int32_t* ox; const int32_t* oy; const int32_t* oz;
    const float* prof;   /* concatenated 1-D Gaussian profiles */
    /* cell -> sources whose box overlaps the cell, ascending source index */
    int32_t cgx, cgy, cgz;
    const int32_t* cell_start; /* [cgx*cgy*cgz + 1] */
    const int32_t* cell_items;
    int32_t kind;        /* VS_SPECTRAL: noise + compact sources; VS_NBODY: no noise, extended halos on zero */
} vs_cube;

#define VS_SPECTRAL 0
#define VS_NBODY 1

/* 64-bit finaliser (splitmix64 constants). Counter-based: any index, any order. */
VS_HD uint64_t vs_mix64(uint64_t x) {
    x += 0x9E3779B97F4A7C15ULL;
    x = (x ^ (x >> 30)) * 0xBF58476D1CE4E5B9ULL;
    x = (x ^ (x >> 27)) * 0x94D049BB133111EBULL;
    return x ^ (x >> 31);
}

VS_HD uint64_t vs_hash2(uint64_t seed, uint64_t idx) {
    return vs_mix64(seed ^ vs_mix64(idx));
}

/* ln((k + 1/2) / 2^32) for a 32-bit k, from IEEE-rounded steps only. */
VS_HD double vs_log01(uint32_t k) {
    uint64_t n = 2ULL * (uint64_t)k + 1ULL;      /* u = n / 2^33, n odd, < 2^33 */
    int p = 63 - VS_CLZ64(n);                    /* top bit */
    double m = (double)(int64_t)n;               /* exact */
    /* scale to [1,2): multiply by 2^-p (exact) */
    double sc = 1.0;
    {
        /* 2^-p built by exact halvings of a table-free constant */
        uint64_t bits = (uint64_t)(1023 - p) << 52;
#if defined(__CUDA_ARCH__)
        sc = __longlong_as_double((long long)bits);
#else
        union { uint64_t u; double d; } cv; cv.u = bits; sc = cv.d;
#endif
    }
    m = VS_DMUL(m, sc);
    int e = p - 33;
    if (m > 1.4142135623730951) { m = VS_DMUL(m, 0.5); e += 1; }
    double s = VS_DDIV(VS_DADD(m, -1.0), VS_DADD(m, 1.0));
    double z = VS_DMUL(s, s);
    double q = 1.0 / 21.0;
    q = VS_FMA(q, z, 1.0 / 19.0);
    q = VS_FMA(q, z, 1.0 / 17.0);
    q = VS_FMA(q, z, 1.0 / 15.0);
    q = VS_FMA(q, z, 1.0 / 13.0);
    q = VS_FMA(q, z, 1.0 / 11.0);
    q = VS_FMA(q, z, 1.0 / 9.0);
    q = VS_FMA(q, z, 1.0 / 7.0);
    q = VS_FMA(q, z, 1.0 / 5.0);
    q = VS_FMA(q, z, 1.0 / 3.0);
    q = VS_FMA(q, z, 1.0);
    double two_s = VS_DADD(s, s);
    return VS_FMA((double)e, 0.6931471805599453, VS_DMUL(two_s, q));
}

/* cos(2*pi*j/2^32): exact octant reduction on the integer, Taylor on [0,pi/4]. */
VS_HD double vs_cos_turn(uint32_t j) {
    uint32_t oct = j >> 29;
    uint32_t r = j & 0x1FFFFFFFu;
    uint32_t rr = (oct & 1u) ? (0x20000000u - r) : r;
    double x = VS_DMUL((double)rr, 1.4629180792671596e-09); /* pi / 2^31 */
    double z = VS_DMUL(x, x);
    /* cos: 1 - z/2 + z^2/24 - ... to z^7 */
    double c = -1.0 / 87178291200.0;
    c = VS_FMA(c, z, 1.0 / 479001600.0);
    c = VS_FMA(c, z, -1.0 / 3628800.0);
    c = VS_FMA(c, z, 1.0 / 40320.0);
    c = VS_FMA(c, z, -1.0 / 720.0);
    c = VS_FMA(c, z, 1.0 / 24.0);
    c = VS_FMA(c, z, -0.5);
    c = VS_FMA(c, z, 1.0);
    /* sin: x (1 - z/6 + z^2/120 - ... to z^6) */
    double s = 1.0 / 6227020800.0;
    s = VS_FMA(s, z, -1.0 / 39916800.0);
    s = VS_FMA(s, z, 1.0 / 362880.0);
    s = VS_FMA(s, z, -1.0 / 5040.0);
    s = VS_FMA(s, z, 1.0 / 120.0);
    s = VS_FMA(s, z, -1.0 / 6.0);
    s = VS_FMA(s, z, 1.0);
    s = VS_DMUL(s, x);
    switch (oct) {
        case 0: case 7: return c;
        case 1: case 6: return s;
        case 2: case 5: return -s;
        default: return -c;
    }
}

/* One N(0,1) draw per index (Box-Muller, cosine branch), rounded to float32. */
VS_HD float vs_noise(uint64_t seed, uint64_t idx) {
    uint64_t h = vs_hash2(seed, idx);
    double lg = vs_log01((uint32_t)(h >> 32));
    double r = VS_DSQRT(VS_DMUL(-2.0, lg));
    double c = vs_cos_turn((uint32_t)(h & 0xFFFFFFFFu));
    return (float)VS_DMUL(r, c);
}

/* The synthetic cube's voxel (x fastest, z = spectral axis). */
VS_HD float vs_voxel(const vs_cube* c, int64_t x, int64_t y, int64_t z) {
    uint64_t idx = (uint64_t)((z * c->ny + y) * c->nx + x);
    float v = c->kind == VS_NBODY ? 0.0f : vs_noise(c->seed, idx);
    if (c->nsrc > 0) {
        int64_t cell = ((z / VS_CELL) * c->cgy + (y / VS_CELL)) * c->cgx + (x / VS_CELL);
        int32_t b = c->cell_start[cell], e = c->cell_start[cell + 1];
        for (int32_t i = b; i < e; ++i) {
            int32_t s = c->cell_items[i];
            int64_t dx = x - c->x0[s], dy = y - c->y0[s], dz = z - c->z0[s];
            if (dx >= 0 && dx < c->lx[s] && dy >= 0 && dy < c->ly[s] && dz >= 0 && dz < c->lz[s]) {
                float w = VS_FMUL(c->peak[s], c->prof[c->ox[s] + dx]);
                w = VS_FMUL(w, c->prof[c->oy[s] + dy]);
                w = VS_FMUL(w, c->prof[c->oz[s] + dz]);
                v = VS_FADD(v, w);
            }
        }
    }
    if (c->ramp != 0.0) {
        double g = VS_DMUL(c->ramp, VS_DDIV(VS_DADD((double)z, 0.5), (double)c->nz));
        v = VS_FADD(v, (float)g);
    }
    return v;
}

/* c4 compositing layers: premultiplied RGBA, alpha ~ U[0,1), rgb = alpha * U[0,1). */
VS_HD void vs_layer_pixel(uint64_t seed, uint64_t layer, uint64_t pix, float out[4]) {
    uint64_t h0 = vs_hash2(seed + 0x1000ULL + layer, 2 * pix);
    uint64_t h1 = vs_hash2(seed + 0x1000ULL + layer, 2 * pix + 1);
    const float k = 5.9604644775390625e-08f; /* 2^-24 */
    float a = VS_FMUL((float)(uint32_t)(h0 >> 40), k);
    float r = VS_FMUL((float)(uint32_t)(h0 & 0xFFFFFFu), k);
    float g = VS_FMUL((float)(uint32_t)(h1 >> 40), k);
    float b = VS_FMUL((float)(uint32_t)(h1 & 0xFFFFFFu), k);
    out[0] = VS_FMUL(a, r); out[1] = VS_FMUL(a, g); out[2] = VS_FMUL(a, b); out[3] = a;
}

#endif /* VR_SYNTH_H */
