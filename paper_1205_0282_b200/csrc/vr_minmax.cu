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
    const int slot_b = vr_slot_index(g, b);
    if (slot_b < 0) return; /* not held by this part (row f3): its table entry stays (+inf, -inf) */
    const float* __restrict__ base = bricks + (long long)slot_b * g.slot;
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

/* ------------------------------------------------------------------------------------------
 * Macro-cells (empty-space skipping inside a brick, R19). A brick's padded cells are cut into
 * 8x8x8 macro-cells (4x4x2 layout: 2x2x4 micro-tiles = 16 whole lines). A sample whose base
 * cell lies in macro-cell m reads cells 8m .. 8m+8 per axis only, so cell_mm[b][m] is the
 * (min, max) over that 9x9x9 block (the macro-cell plus one layer on its high sides): it
 * bounds everything such a sample can interpolate between. A macro-cell is flagged
 * TRANSPARENT for the current transfer function with R16's rule on that range; the ray-cast
 * kernels then skip the samples based in it: their opacity is exactly zero, so the frame does
 * not change by a bit.
 * ---------------------------------------------------------------------------------------- */
__global__ void __launch_bounds__(256)
vr_cell_minmax_kernel(VrGrid g, const float* __restrict__ bricks, float2* __restrict__ cell_mm, int nc0, int nc1, int nc2) {
    /* one warp per macro-cell: 16 micro-tiles x 8 rows = 128 float4 words, 4 per lane */
    const int b = blockIdx.y;
    int bc[3], lo[3], hi[3];
    vr_brick_coords(g, b, bc);
    vr_brick_core(g, bc, lo, hi);
    const int ex = hi[0] - lo[0] + 2 * g.ghost, ey = hi[1] - lo[1] + 2 * g.ghost, ez = hi[2] - lo[2] + 2 * g.ghost;
    const int slot_b = vr_slot_index(g, b);
    if (slot_b < 0) return; /* the macro-cell tables have one row per held brick, by slot */
    const float* __restrict__ base = bricks + (long long)slot_b * g.slot;
    const int lane = threadIdx.x & 31, ncell = nc0 * nc1 * nc2;
    for (int m = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5); m < ncell; m += gridDim.x * (blockDim.x >> 5)) {
        const int m2 = m / (nc0 * nc1), rem = m - m2 * (nc0 * nc1), m1 = rem / nc0, m0 = rem - m1 * nc0;
        float mn = INFINITY, mx = -INFINITY;
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            const int w = lane + 32 * q;           /* word of the macro-cell: tile (w >> 3), row (w & 7) */
            const int t = w >> 3, r = w & 7;
            const int tx = (m0 << 1) + (t & 1), ty = (m1 << 1) + ((t >> 1) & 1), tz = (m2 << 2) + (t >> 2);
            const int i = tx << 2, j = (ty << 2) + (r & 3), k = (tz << 1) + (r >> 2);
            if (tx < g.nt[0] && ty < g.nt[1] && tz < g.nt[2] && i < ex && j < ey && k < ez) {
                const long long word = ((long long)((tz * g.nt[1] + ty) * g.nt[0] + tx) << 3) + r;
                const float4 v = __ldcs(reinterpret_cast<const float4*>(base) + word);
                mn = fminf(mn, v.x), mx = fmaxf(mx, v.x);
                if (i + 1 < ex) mn = fminf(mn, v.y), mx = fmaxf(mx, v.y);
                if (i + 2 < ex) mn = fminf(mn, v.z), mx = fmaxf(mx, v.z);
                if (i + 3 < ex) mn = fminf(mn, v.w), mx = fmaxf(mx, v.w);
            }
        }
        /* the layer on the high sides: planes x = 8 (9x9), y = 8 (8x9), z = 8 (8x8) of the 9x9x9 block */
        for (int h = lane; h < 217; h += 32) {
            int a, c, d;
            if (h < 81) a = 8, c = h % 9, d = h / 9;
            else if (h < 153) a = (h - 81) & 7, c = 8, d = (h - 81) >> 3;
            else a = (h - 153) & 7, c = (h - 153) >> 3, d = 8;
            const int i = (m0 << 3) + a, j = (m1 << 3) + c, k = (m2 << 3) + d;
            if (i < ex && j < ey && k < ez) {
                const float x = __ldg(base + vr_cell_offset(g, i, j, k));
                mn = fminf(mn, x), mx = fmaxf(mx, x);
            }
        }
        for (int o = 16; o > 0; o >>= 1) {
            mn = fminf(mn, __shfl_xor_sync(0xffffffffu, mn, o));
            mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, o));
        }
        if (lane == 0) cell_mm[(long long)slot_b * ncell + m] = make_float2(mn + 0.0f, mx + 0.0f);
    }
}

/* bits[b][m] = 1 iff macro-cell m of brick b is transparent under the LUT (R19). One thread per cell. */
__global__ void __launch_bounds__(256)
vr_cell_flags_kernel(const float2* __restrict__ cell_mm, unsigned* __restrict__ bits, int nbricks, int nc0, int nc1, int nc2,
                     int words_per_brick, VrLut lut) {
    __shared__ unsigned short nz_prefix[VR_MAX_LUT + 1];
    for (int i = threadIdx.x; i < lut.n; i += blockDim.x) nz_prefix[i + 1] = lut.base[i].w != 0.0f ? 1 : 0;
    __syncthreads();
    if (threadIdx.x == 0) {
        nz_prefix[0] = 0;
        for (int i = 1; i <= lut.n; ++i) nz_prefix[i] = (unsigned short)(nz_prefix[i] + nz_prefix[i - 1]);
    }
    __syncthreads();
    const int ncell = nc0 * nc1 * nc2;
    const long long total = (long long)nbricks * words_per_brick * 32;
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < total; t += (long long)gridDim.x * blockDim.x) {
        const int b = (int)(t / (words_per_brick * 32)), m = (int)(t - (long long)b * words_per_brick * 32);
        bool transparent = false;
        if (m < ncell) {
            const float2 rr = cell_mm[(long long)b * ncell + m];
            const float mn = rr.x, mx = rr.y;
            if (mn <= mx) { /* R16's entry range in float32 */
                const float ulo = __saturatef(__fmul_rn(__fsub_rn(mn, lut.vmin), lut.inv_range));
                const float uhi = __saturatef(__fmul_rn(__fsub_rn(mx, lut.vmin), lut.inv_range));
                const int i0 = max(min((int)__fmul_rn(ulo, lut.scale), lut.nm2) - 1, 0);
                const int i1 = min(min((int)__fmul_rn(uhi, lut.scale), lut.nm2) + 2, lut.n - 1);
                transparent = nz_prefix[i1 + 1] == nz_prefix[i0];
            }
        }
        const unsigned word = __ballot_sync(0xffffffffu, transparent);
        if ((threadIdx.x & 31) == 0) bits[t >> 5] = word;
    }
}

/* ------------------------------------------------------------------------------------------
 * Both tables from ONE streaming read of the store (one min/max task after the data is loaded).
 * A warp takes a macro-cell: its 16 micro-tiles = 128 float4 words, 4 per lane (lane -> tile column tx, tile row ty and
 * row r of the micro-tile are fixed, the 4 words differ in tile layer tz). The 9x9x9 block R19 asks for is the macro-
 * cell's own 8x8x8 cells plus the FIRST planes of its high-side neighbours; seen from the neighbour, its planes x = 0,
 * y = 0, z = 0, their three common edges and the corner belong to the blocks of the macro-cells on its low sides. So a
 * warp reduces eight ranges - own cells, three faces, three edges, corner - with REDUX on the order-preserving integer
 * encoding (16 instructions) and merges each into the table entry of the macro-cell it belongs to with integer atomics
 * (distinct addresses, absorbed by L2). The brick's range is the union of its macro-cells' own-cell ranges: kept in
 * registers across a CTA's macro-cells, two atomics per CTA. No cell is read twice; the halo reads that cost the two-pass
 * version 1.47x the store's bytes are gone.
 * ---------------------------------------------------------------------------------------- */
__global__ void vr_range_init_kernel(int2* __restrict__ cell_enc, long long ncells, int2* __restrict__ brick_enc, int nbricks) {
    const int2 e = make_int2(mm_encode(INFINITY), mm_encode(-INFINITY));
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < ncells; i += (long long)gridDim.x * blockDim.x) cell_enc[i] = e;
    if (blockIdx.x == 0)
        for (int b = threadIdx.x; b < nbricks; b += blockDim.x) brick_enc[b] = e;
}

__device__ __forceinline__ void range_merge(int2* __restrict__ p, int mn, int mx) {
    if (mn <= mx) {
        atomicMin(&p->x, mn);
        atomicMax(&p->y, mx);
    }
}

__global__ void __launch_bounds__(256)
vr_range_kernel(VrGrid g, const float* __restrict__ bricks, int2* __restrict__ cell_enc, const int4* __restrict__ slot_ext, int nc0,
                int nc1, int nc2) {
    /* grid (1, rows x layers of macro-cells, slots): a CTA takes one row of macro-cells, warp w the macro-cells
     * m0 = w, w + 8, ... of it: the per-row index arithmetic is paid once per warp, the words of the next macro-cell are
     * 16 float4 further on (the first version, a grid-stride loop over all macro-cells with two divisions per cell and
     * eight predicated accumulators, was ALU-bound at 554 instructions per macro-cell) */
    const int slot_b = blockIdx.z;
    const int4 ext = __ldg(slot_ext + slot_b); /* padded extent of the brick in this slot (x, y, z) */
    const int ex = ext.x, ey = ext.y, ez = ext.z;
    const int lane = threadIdx.x & 31;
    const int m2 = blockIdx.y / nc1, m1 = blockIdx.y - m2 * nc1;
    const float4* __restrict__ base = reinterpret_cast<const float4*>(bricks + (long long)slot_b * g.slot);
    const int tcol = (lane >> 3) & 1, trow = lane >> 4, r = lane & 7;
    const int jl = (trow << 2) + (r & 3); /* the lane's y inside the macro-cell; x = 4 tcol .. 4 tcol + 3; z = 2 q + (r >> 2) */
    const int ty = (m1 << 1) + trow;
    const bool row_ok = ty < g.nt[1] && (m1 << 3) + jl < ey;
    bool okz[4];
#pragma unroll
    for (int q = 0; q < 4; ++q) okz[q] = row_ok && (m2 << 2) + q < g.nt[2] && (((m2 << 2) + q) << 1) + (r >> 2) < ez;
    const long long wrow = ((long long)(((m2 << 2) * g.nt[1] + ty) * g.nt[0]) << 3) + r, wz = (long long)g.nt[1] * g.nt[0] << 3;
    const bool x0 = tcol == 0, y0 = jl == 0, z0 = r < 4;
    const int E_HI = mm_encode(INFINITY), E_LO = mm_encode(-INFINITY);
    int2* __restrict__ cells = cell_enc + (long long)slot_b * (nc0 * nc1 * nc2);
    /* which range this lane merges (lanes 0..7: own, -x, -y, -z, -x-y, -x-z, -y-z, -x-y-z) and into which macro-cell */
    const int dx = (0xB2 >> (lane & 7)) & 1, dy = (0xD4 >> (lane & 7)) & 1, dz = (0xE8 >> (lane & 7)) & 1;
    const bool merges = lane < 8 && m1 - dy >= 0 && m2 - dz >= 0;
    int2* __restrict__ target = cells + ((m2 - dz) * nc1 + (m1 - dy)) * nc0 - dx;
    for (int m0 = threadIdx.x >> 5; m0 < nc0; m0 += blockDim.x >> 5) {
        const int tx = (m0 << 1) + tcol, i = tx << 2;
        const bool col_ok = tx < g.nt[0] && i < ex;
        const float4* __restrict__ p = base + (wrow + ((long long)tx << 3));
        float4 v[4];
#pragma unroll
        for (int q = 0; q < 4; ++q) /* all four loads first */
            if (col_ok && okz[q]) v[q] = __ldcs(p + q * wz);
        /* per lane: A = range of its words (own cells), B = range of their first elements (the column x = 4 tcol), and
         * both restricted to the plane z = 0 (word q = 0 of the lanes with r < 4) */
        float amn = INFINITY, amx = -INFINITY, bmn = INFINITY, bmx = -INFINITY, azmn = INFINITY, azmx = -INFINITY, bzmn = INFINITY,
              bzmx = -INFINITY;
        const bool full = i + 3 < ex;
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            if (!(col_ok && okz[q])) continue;
            float wmn, wmx; /* cells beyond the brick's extent are left out */
            if (full) {
                wmn = fminf(fminf(v[q].x, v[q].y), fminf(v[q].z, v[q].w));
                wmx = fmaxf(fmaxf(v[q].x, v[q].y), fmaxf(v[q].z, v[q].w));
            } else {
                wmn = wmx = v[q].x;
                if (i + 1 < ex) wmn = fminf(wmn, v[q].y), wmx = fmaxf(wmx, v[q].y);
                if (i + 2 < ex) wmn = fminf(wmn, v[q].z), wmx = fmaxf(wmx, v[q].z);
            }
            amn = fminf(amn, wmn), amx = fmaxf(amx, wmx);
            bmn = fminf(bmn, v[q].x), bmx = fmaxf(bmx, v[q].x);
            if (q == 0 && z0) /* through fminf / fmaxf: a NaN (blanked) cell must not become a bound (R14) */
                azmn = fminf(azmn, wmn), azmx = fmaxf(azmx, wmx), bzmn = fminf(bzmn, v[q].x), bzmx = fmaxf(bzmx, v[q].x);
        }
        /* the eight ranges: 0 own cells, 1 x = 0, 2 y = 0, 3 z = 0, 4 x = y = 0, 5 x = z = 0, 6 y = z = 0, 7 corner; a lane
         * contributes to a face only if it holds cells of it (lane-constant conditions). fminf / fmaxf ignored NaN
         * voxels (R14); an untouched range stays (+inf, -inf) */
        const int eamn = mm_encode(amn), eamx = mm_encode(amx), ebmn = mm_encode(bmn), ebmx = mm_encode(bmx);
        const int eazmn = mm_encode(azmn), eazmx = mm_encode(azmx), ebzmn = mm_encode(bzmn), ebzmx = mm_encode(bzmx);
        int smn = E_HI, smx = E_LO, t;
#define VR_RANGE(c, vmn, vmx)                                        \
    t = __reduce_min_sync(0xffffffffu, (vmn)); if (lane == (c)) smn = t; \
    t = __reduce_max_sync(0xffffffffu, (vmx)); if (lane == (c)) smx = t;
        VR_RANGE(0, eamn, eamx)
        VR_RANGE(1, x0 ? ebmn : E_HI, x0 ? ebmx : E_LO)
        VR_RANGE(2, y0 ? eamn : E_HI, y0 ? eamx : E_LO)
        VR_RANGE(3, eazmn, eazmx)
        VR_RANGE(4, x0 && y0 ? ebmn : E_HI, x0 && y0 ? ebmx : E_LO)
        VR_RANGE(5, x0 ? ebzmn : E_HI, x0 ? ebzmx : E_LO)
        VR_RANGE(6, y0 ? eazmn : E_HI, y0 ? eazmx : E_LO)
        VR_RANGE(7, x0 && y0 ? ebzmn : E_HI, x0 && y0 ? ebzmx : E_LO)
#undef VR_RANGE
        if (merges && m0 - dx >= 0) range_merge(target + m0, smn, smx);
    }
}

/* Decode the macro-cell table in place (int2 -> float2, -0 -> +0 as the two-pass version did) and reduce each brick's
 * entries to the brick's range: the union of the 9x9x9 blocks of a brick's macro-cells is the brick's padded cells. */
__global__ void __launch_bounds__(256)
vr_range_finish_cells_kernel(VrGrid g, int2* __restrict__ cell_enc, int ncell, int2* __restrict__ brick_enc) {
    const int b = blockIdx.y;
    const int slot_b = vr_slot_index(g, b);
    if (slot_b < 0) return;
    int2* __restrict__ cells = cell_enc + (long long)slot_b * ncell;
    int bmn = mm_encode(INFINITY), bmx = mm_encode(-INFINITY);
    for (int m = blockIdx.x * blockDim.x + threadIdx.x; m < ncell; m += gridDim.x * blockDim.x) {
        const int2 e = cells[m];
        if (e.x <= e.y) bmn = min(bmn, e.x), bmx = max(bmx, e.y);
        reinterpret_cast<float2*>(cells)[m] = make_float2(mm_decode(e.x), mm_decode(e.y));
    }
    bmn = __reduce_min_sync(0xffffffffu, bmn);
    bmx = __reduce_max_sync(0xffffffffu, bmx);
    __shared__ int s_mn[8], s_mx[8];
    if ((threadIdx.x & 31) == 0) s_mn[threadIdx.x >> 5] = bmn, s_mx[threadIdx.x >> 5] = bmx;
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int w = 1; w < (int)(blockDim.x >> 5); ++w) bmn = min(bmn, s_mn[w]), bmx = max(bmx, s_mx[w]);
        range_merge(brick_enc + b, bmn, bmx);
    }
}

cudaError_t vr_launch_ranges(const VrGrid& grid, const float* bricks, int2* enc, float2* table, float2* cell_mm, const int nc[3],
                             const int4* slot_ext, cudaStream_t st) {
    const int ncell = nc[0] * nc[1] * nc[2];
    const long long total = (long long)ncell * grid.nown;
    if ((long long)nc[1] * nc[2] > 65535 || grid.nbricks > 65535) return cudaErrorInvalidValue;
    int2* cell_enc = reinterpret_cast<int2*>(cell_mm);
    vr_range_init_kernel<<<148 * 8, 256, 0, st>>>(cell_enc, total, enc, grid.nbricks);
    vr_range_kernel<<<dim3(1u, (unsigned)(nc[1] * nc[2]), (unsigned)grid.nown), 256, 0, st>>>(grid, bricks, cell_enc, slot_ext, nc[0],
                                                                                               nc[1], nc[2]);
    int fx = (ncell + 256 * 8 - 1) / (256 * 8);
    if (fx > 64) fx = 64;
    vr_range_finish_cells_kernel<<<dim3((unsigned)fx, (unsigned)grid.nbricks), 256, 0, st>>>(grid, cell_enc, ncell, enc);
    vr_minmax_finish_kernel<<<1, 256, 0, st>>>(enc, grid.nbricks, table);
    return cudaGetLastError();
}

cudaError_t vr_launch_cell_minmax(const VrGrid& grid, const float* bricks, float2* cell_mm, const int nc[3], cudaStream_t st) {
    const long long ncell = (long long)nc[0] * nc[1] * nc[2];
    long long bx = (ncell + 7) / 8;
    if (bx > 4096) bx = 4096;
    vr_cell_minmax_kernel<<<dim3((unsigned)bx, grid.nbricks), 256, 0, st>>>(grid, bricks, cell_mm, nc[0], nc[1], nc[2]);
    return cudaGetLastError();
}

cudaError_t vr_launch_cell_flags(const float2* cell_mm, unsigned* bits, int nbricks, const int nc[3], int words_per_brick,
                                 const VrLut& lut, cudaStream_t st) {
    const long long total = (long long)nbricks * words_per_brick * 32;
    long long blocks = (total + 255) / 256;
    if (blocks > 148 * 16) blocks = 148 * 16;
    vr_cell_flags_kernel<<<(unsigned)blocks, 256, 0, st>>>(cell_mm, bits, nbricks, nc[0], nc[1], nc[2], words_per_brick, lut);
    return cudaGetLastError();
}

__global__ void __launch_bounds__(256)
vr_cell_count_empty_kernel(const float2* __restrict__ cell_mm, long long ncells, const float2* __restrict__ global_mm,
                           unsigned long long* __restrict__ count) {
    const float lo = global_mm->x;
    unsigned c = 0;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < ncells; i += (long long)gridDim.x * blockDim.x) {
        const float2 r = cell_mm[i];
        c += (r.x == lo && r.y == lo) ? 1u : 0u;
    }
    for (int o = 16; o > 0; o >>= 1) c += __shfl_xor_sync(0xffffffffu, c, o);
    if ((threadIdx.x & 31) == 0 && c) atomicAdd(count, (unsigned long long)c);
}

cudaError_t vr_launch_cell_count_empty(const float2* cell_mm, long long ncells, const float2* global_mm, unsigned long long* count,
                                       cudaStream_t st) {
    vr_cell_count_empty_kernel<<<148 * 8, 256, 0, st>>>(cell_mm, ncells, global_mm, count);
    return cudaGetLastError();
}


/* R20 (vii): the mean range of the macro-cells that hold finite data - the scale of the voxel-to-voxel differences the
 * texture filter's error is proportional to. stat[0] += sum of (max - min), stat[1] += number of such cells. */
__global__ void __launch_bounds__(256)
vr_cell_range_sum_kernel(const float2* __restrict__ cell_mm, long long ncells, double* __restrict__ stat) {
    double sum = 0.0, cnt = 0.0;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < ncells; i += (long long)gridDim.x * blockDim.x) {
        const float2 r = cell_mm[i];
        const float d = r.y - r.x;
        if (d >= 0.0f && d < INFINITY) sum += (double)d, cnt += 1.0;
    }
    for (int o = 16; o > 0; o >>= 1) sum += __shfl_xor_sync(0xffffffffu, sum, o), cnt += __shfl_xor_sync(0xffffffffu, cnt, o);
    if ((threadIdx.x & 31) == 0 && cnt > 0.0) {
        atomicAdd(stat, sum);
        atomicAdd(stat + 1, cnt);
    }
}

cudaError_t vr_launch_cell_range_sum(const float2* cell_mm, long long ncells, double* stat, cudaStream_t st) {
    vr_cell_range_sum_kernel<<<148 * 8, 256, 0, st>>>(cell_mm, ncells, stat);
    return cudaGetLastError();
}
