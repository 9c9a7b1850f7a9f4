/*
 * vr_minmax.cu -- the data range of the brick store.
 *
 * PAPER.md:146 (sec. 2.3.1): "An independent task to determine the local minimum and maximum
 * starts when the data is loaded into the GPU memory"; :152 the march may stop at "the maximum
 * pixel value (defined by the global maximum of the data)". Local = per brick, over the
 * brick's ghost-padded cells: every value a sample of that brick can interpolate between.
 * The per-view set-up uses the table to skip bricks the transfer function makes transparent
 * (R16) and the ray-cast kernel stops MIP rays at the global maximum.
 *
 * One streaming pass over the store after an upload (not per frame): grid (x, brick), every
 * thread reads 16-byte words in memory order (4x4x2 layout: one x-row of a micro-tile, the
 * cells beyond the brick's extent masked out), min/max by warp shuffles and shared memory, one
 * pair of atomics per CTA on an order-preserving integer encoding of the floats. A second one-CTA kernel
 * decodes the table and reduces it to the range of the whole volume.
 */
#include <math.h>

#include "vr_view.cuh"

/* float -> int, monotone: a < b  <=>  enc(a) < enc(b) (no NaNs: R14) */
__device__ __forceinline__ int mm_encode(float f) {
    const int i = __float_as_int(f);
    return i >= 0 ? i : i ^ 0x7fffffff;
}
__device__ __forceinline__ float mm_decode(int i) { return __int_as_float(i >= 0 ? i : i ^ 0x7fffffff) + 0.0f; }

__global__ void vr_minmax_init_kernel(int2* __restrict__ enc, int n) {
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b < n) enc[b] = make_int2(mm_encode(INFINITY), mm_encode(-INFINITY));
}

template <bool TILE442>
__global__ void __launch_bounds__(256)
vr_brick_minmax_kernel(VrGrid g, const float* __restrict__ bricks, int2* __restrict__ enc) {
    const int b = blockIdx.y;
    int bc[3], lo[3], hi[3];
    vr_brick_coords(g, b, bc);
    vr_brick_core(g, bc, lo, hi);
    const int ex = hi[0] - lo[0] + 2 * g.ghost, ey = hi[1] - lo[1] + 2 * g.ghost, ez = hi[2] - lo[2] + 2 * g.ghost;
    const float* __restrict__ base = bricks + (long long)b * g.slot;
    float mn = INFINITY, mx = -INFINITY;
    if (TILE442) {
        /* word u of the slot = row r = u & 7 (lj = r & 3, lk = r >> 2) of tile u >> 3 */
        const unsigned nt0 = (unsigned)g.nt[0], nt01 = nt0 * (unsigned)g.nt[1];
        const unsigned words = (unsigned)(g.slot >> 2);
        for (unsigned u = blockIdx.x * blockDim.x + threadIdx.x; u < words; u += gridDim.x * blockDim.x) {
            const unsigned t = u >> 3, r = u & 7u;
            const unsigned tz = t / nt01, rem = t - tz * nt01, ty = rem / nt0, tx = rem - ty * nt0;
            const int i = (int)(tx << 2), j = (int)(ty << 2) + (int)(r & 3u), k = (int)(tz << 1) + (int)(r >> 2);
            if (j < ey && k < ez && i < ex) {
                const float4 q = __ldcs(reinterpret_cast<const float4*>(base) + u);
                mn = fminf(mn, q.x), mx = fmaxf(mx, q.x);
                if (i + 1 < ex) mn = fminf(mn, q.y), mx = fmaxf(mx, q.y);
                if (i + 2 < ex) mn = fminf(mn, q.z), mx = fmaxf(mx, q.z);
                if (i + 3 < ex) mn = fminf(mn, q.w), mx = fmaxf(mx, q.w);
            }
        }
    } else {
        /* any separable layout: one warp per padded (j,k) row, lanes along i */
        const int rows = ey * ez, lane = threadIdx.x & 31, wpb = blockDim.x >> 5;
        for (int row = blockIdx.x * wpb + (threadIdx.x >> 5); row < rows; row += gridDim.x * wpb) {
            const int j = row % ey, k = row / ey;
            const unsigned oyz = vr_axis_offset(g.ax[1], j) + vr_axis_offset(g.ax[2], k);
            for (int i = lane; i < ex; i += 32) {
                const float x = __ldcs(base + (oyz + vr_axis_offset(g.ax[0], i)));
                mn = fminf(mn, x), mx = fmaxf(mx, x);
            }
        }
    }
    for (int o = 16; o > 0; o >>= 1) {
        mn = fminf(mn, __shfl_xor_sync(0xffffffffu, mn, o));
        mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, o));
    }
    /* one pair of atomics per CTA: same-address atomics serialise in L2 (~2 ns each) */
    __shared__ float s_mn[8], s_mx[8];
    if ((threadIdx.x & 31) == 0) s_mn[threadIdx.x >> 5] = mn, s_mx[threadIdx.x >> 5] = mx;
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int w = 1; w < (int)(blockDim.x >> 5); ++w) mn = fminf(mn, s_mn[w]), mx = fmaxf(mx, s_mx[w]);
        if (mn <= mx) {
            atomicMin(&enc[b].x, mm_encode(mn));
            atomicMax(&enc[b].y, mm_encode(mx));
        }
    }
}

/* table[b] = (min, max) of brick b; table[nbricks] = the range of the whole volume */
__global__ void __launch_bounds__(256)
vr_minmax_finish_kernel(const int2* __restrict__ enc, int n, float2* __restrict__ table) {
    __shared__ float s_mn[8], s_mx[8];
    float mn = INFINITY, mx = -INFINITY;
    for (int b = threadIdx.x; b < n; b += blockDim.x) {
        const int2 e = enc[b];
        const float lo = mm_decode(e.x), hi = mm_decode(e.y);
        table[b] = make_float2(lo, hi);
        mn = fminf(mn, lo), mx = fmaxf(mx, hi);
    }
    for (int o = 16; o > 0; o >>= 1) {
        mn = fminf(mn, __shfl_xor_sync(0xffffffffu, mn, o));
        mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, o));
    }
    if ((threadIdx.x & 31) == 0) s_mn[threadIdx.x >> 5] = mn, s_mx[threadIdx.x >> 5] = mx;
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int w = 1; w < 8; ++w) mn = fminf(mn, s_mn[w]), mx = fmaxf(mx, s_mx[w]);
        table[n] = make_float2(mn, mx);
    }
}

cudaError_t vr_launch_minmax(const VrGrid& grid, const float* bricks, int2* enc, float2* table, cudaStream_t st) {
    vr_minmax_init_kernel<<<(grid.nbricks + 255) / 256, 256, 0, st>>>(enc, grid.nbricks);
    const bool t442 = grid.layout == VR_LAYOUT_TILED && grid.tl[0] == 2 && grid.tl[1] == 2 && grid.tl[2] == 1 &&
                      grid.ml[0] == 0 && grid.ml[1] == 0 && grid.ml[2] == 0;
    /* enough CTAs per brick to fill the machine several times over, few enough to keep the atomics rare */
    long long per_brick = t442 ? (grid.slot / 4 + 256 * 32 - 1) / (256 * 32) : ((long long)grid.P * grid.P + 7) / 8;
    if (per_brick > 1024) per_brick = 1024;
    if (per_brick < 1) per_brick = 1;
    const dim3 gr((unsigned)per_brick, grid.nbricks);
    if (t442) vr_brick_minmax_kernel<true><<<gr, 256, 0, st>>>(grid, bricks, enc);
    else vr_brick_minmax_kernel<false><<<gr, 256, 0, st>>>(grid, bricks, enc);
    vr_minmax_finish_kernel<<<1, 256, 0, st>>>(enc, grid.nbricks, table);
    return cudaGetLastError();
}
