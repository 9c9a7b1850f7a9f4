/*
 * vr_bricks.cu -- the brick store.
 *
 * PAPER.md:105,113 (sec. 2.1): the cube is split into sub-cubes that are rendered
 * independently; :136 (sec. 2.3.1) partitioning; :146 the data is moved into GPU memory once,
 * before rendering. The paper keeps each sub-cube in texture memory (:150); here a brick is a
 * ghost-padded float32 array in HBM, either x-linear rows or 128-byte 3-D micro-tiles
 * (DESIGN.md "Data layout" says why).
 *
 * Ghost cells (R3): cell (i,j,k) of brick b holds global voxel clamp(lo_b - ghost + (i,j,k),
 * 0, n-1), so every tri-linear fetch of a sample the brick owns stays inside the brick and
 * the volume boundary is edge-replicated.
 *
 * Upload is a gather. LINEAR: one warp per padded row of one brick, lanes along x (coalesced
 * writes, coalesced reads except at the two replicated ends). TILED: one CTA per row of
 * micro-tiles, source rows staged in shared memory so that both the reads and the writes are
 * whole 128-byte lines. A cell is written iff its clamped global index lies in the uploaded
 * box, which makes z-slab uploads of a ~100 GB cube work.
 */
#include "vr_view.cuh"

/* range [a0,a1) of padded indices i in [0,ext) with clamp(lo - ghost + i, 0, n-1) in [c0,c1) */
__device__ __forceinline__ void padded_range(int lo, int ghost, int ext, int n, int c0, int c1, int& a0, int& a1) {
    /* global index x(i) = clamp(lo - ghost + i, 0, n-1) is non-decreasing in i */
    const int base = lo - ghost;
    /* first i with x(i) >= c0 */
    int f0 = c0 - base;              /* unclamped solution */
    if (c0 <= 0) f0 = 0;             /* clamped-low cells map to 0 >= c0 */
    if (c0 > n - 1) f0 = ext;        /* never reached */
    /* first i with x(i) >= c1 */
    int f1 = c1 - base;
    if (c1 <= 0) f1 = 0;
    if (c1 > n - 1) f1 = ext;
    a0 = min(max(f0, 0), ext);
    a1 = min(max(f1, 0), ext);
}

__global__ void __launch_bounds__(256)
vr_upload_kernel(VrGrid g, float* __restrict__ bricks, const float* __restrict__ src, int x0, int y0, int z0, int sx, int sy,
                 int sz, int b0) {
    const int b = blockIdx.y + b0; /* b0: first brick of the z range the box can touch */
    int bc[3], lo[3], hi[3];
    vr_brick_coords(g, b, bc);
    vr_brick_core(g, bc, lo, hi);
    const int ex = hi[0] - lo[0] + 2 * g.ghost, ey = hi[1] - lo[1] + 2 * g.ghost, ez = hi[2] - lo[2] + 2 * g.ghost;
    int i0, i1, j0, j1, k0, k1;
    padded_range(lo[0], g.ghost, ex, g.n[0], x0, x0 + sx, i0, i1);
    padded_range(lo[1], g.ghost, ey, g.n[1], y0, y0 + sy, j0, j1);
    padded_range(lo[2], g.ghost, ez, g.n[2], z0, z0 + sz, k0, k1);
    if (i1 <= i0 || j1 <= j0 || k1 <= k0) return;
    const int slot_b = vr_slot_index(g, b);
    if (slot_b < 0) return; /* a part handle does not hold this brick (row f3) */
    const int rows = (j1 - j0) * (k1 - k0);
    const int warps_per_block = blockDim.x >> 5, lane = threadIdx.x & 31;
    float* __restrict__ dstb = bricks + (long long)slot_b * g.slot;
    for (int row = blockIdx.x * warps_per_block + (threadIdx.x >> 5); row < rows; row += gridDim.x * warps_per_block) {
        const int j = j0 + row % (j1 - j0), k = k0 + row / (j1 - j0);
        const int gy = min(max(lo[1] - g.ghost + j, 0), g.n[1] - 1), gz = min(max(lo[2] - g.ghost + k, 0), g.n[2] - 1);
        const float* __restrict__ srow = src + ((long long)(gz - z0) * sy + (gy - y0)) * sx;
        float* __restrict__ drow = dstb + ((long long)k * g.P + j) * g.P;
        for (int i = i0 + lane; i < i1; i += 32) {
            const int gx = min(max(lo[0] - g.ghost + i, 0), g.n[0] - 1);
            drow[i] = __ldcs(srow + (gx - x0));
        }
    }
}

/* TILED: a CTA takes groups of TR consecutive rows of micro-tiles (same tile z) of one brick,
 * TR * 2^(tl1+tl2) <= 32 source rows at a time. Phase 1 stages those source rows in shared
 * memory: each warp owns up to 4 rows and keeps 8 coalesced 128-byte reads in flight (lanes
 * along x; the replicated ends re-read one cell). Phase 2 writes the micro-tiles, one warp per
 * tile = one 128-byte line, lane = cell inside the tile. The row pitch is = 4 (mod 32) floats
 * so that the rows x cells a warp gathers fall into different banks. Both sides of the copy
 * move whole lines: an HBM streaming kernel. */
#define UP_ROWS 32 /* staged source rows per group (at most) */

__global__ void __launch_bounds__(256)
vr_upload_tiled_kernel(VrGrid g, float* __restrict__ bricks, const float* __restrict__ src, int x0, int y0, int z0, int sx,
                       int sy, int sz, int pitch, int b0) {
    extern __shared__ float s_rows[];
    const int b = blockIdx.y + b0; /* b0: first brick of the z range the box can touch */
    int bc[3], lo[3], hi[3];
    vr_brick_coords(g, b, bc);
    vr_brick_core(g, bc, lo, hi);
    const int ex = hi[0] - lo[0] + 2 * g.ghost, ey = hi[1] - lo[1] + 2 * g.ghost, ez = hi[2] - lo[2] + 2 * g.ghost;
    int i0, i1, j0, j1, k0, k1;
    padded_range(lo[0], g.ghost, ex, g.n[0], x0, x0 + sx, i0, i1);
    padded_range(lo[1], g.ghost, ey, g.n[1], y0, y0 + sy, j0, j1);
    padded_range(lo[2], g.ghost, ez, g.n[2], z0, z0 + sz, k0, k1);
    if (i1 <= i0 || j1 <= j0 || k1 <= k0) return;
    const int slot_b = vr_slot_index(g, b);
    if (slot_b < 0) return; /* a part handle does not hold this brick (row f3) */
    const int tx0 = i0 >> g.tl[0], tx1 = ((i1 - 1) >> g.tl[0]) + 1, ntx = tx1 - tx0;
    const int ty0 = j0 >> g.tl[1], ty1 = ((j1 - 1) >> g.tl[1]) + 1;
    const int tz0 = k0 >> g.tl[2], tz1 = ((k1 - 1) >> g.tl[2]) + 1;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, nwarps = blockDim.x >> 5;
    const int rbits = g.tl[1] + g.tl[2], nrow = 1 << rbits; /* source rows per tile row */
    const int TR = UP_ROWS >> rbits;                        /* tile rows per group */
    const int ngy = (ty1 - ty0 + TR - 1) / TR, groups = ngy * (tz1 - tz0);
    const int li = lane & ((1 << g.tl[0]) - 1), ljk = lane >> g.tl[0];
    const int lj = ljk & ((1 << g.tl[1]) - 1), lk = ljk >> g.tl[1];
    const int ibase = tx0 << g.tl[0]; /* first staged padded x index */
    float* __restrict__ dstb = bricks + (long long)slot_b * g.slot;
    for (int grp = blockIdx.x; grp < groups; grp += gridDim.x) {
        const int tyg = ty0 + (grp % ngy) * TR, kt = (tz0 + grp / ngy) << g.tl[2];
        const int ntr = min(TR, ty1 - tyg); /* tile rows in this group */
        /* phase 1: rows r = warp, warp + 8, ... of the group; r = (tile row, lk, lj) */
        const float* srow[4];
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            const int r = warp + q * nwarps;
            const int j = ((tyg + (r >> rbits)) << g.tl[1]) + (r & ((1 << g.tl[1]) - 1));
            const int k = kt + ((r >> g.tl[1]) & ((1 << g.tl[2]) - 1));
            srow[q] = NULL;
            if (r < (ntr << rbits) && j >= j0 && j < j1 && k >= k0 && k < k1) {
                const int gy = min(max(lo[1] - g.ghost + j, 0), g.n[1] - 1), gz = min(max(lo[2] - g.ghost + k, 0), g.n[2] - 1);
                srow[q] = src + ((long long)(gz - z0) * sy + (gy - y0)) * sx - x0;
            }
        }
        for (int i = i0 + lane; i < i1; i += 64) {
            float v[4][2];
#pragma unroll
            for (int q = 0; q < 4; ++q)
#pragma unroll
                for (int u = 0; u < 2; ++u) {
                    const int gx = min(max(lo[0] - g.ghost + min(i + 32 * u, i1 - 1), 0), g.n[0] - 1);
                    v[q][u] = srow[q] ? __ldcs(srow[q] + gx) : 0.0f;
                }
#pragma unroll
            for (int q = 0; q < 4; ++q)
#pragma unroll
                for (int u = 0; u < 2; ++u)
                    if (srow[q] && i + 32 * u < i1) s_rows[(warp + q * nwarps) * pitch + (i + 32 * u - ibase)] = v[q][u];
        }
        __syncthreads();
        /* phase 2: tile t of the group = (tile row t / ntx, tile x t % ntx) */
        for (int t = warp; t < ntr * ntx; t += nwarps) {
            const int tr = t / ntx, tx = tx0 + (t - tr * ntx);
            const int i = (tx << g.tl[0]) + li, j = ((tyg + tr) << g.tl[1]) + lj, k = kt + lk;
            if (i >= i0 && i < i1 && j >= j0 && j < j1 && k >= k0 && k < k1)
                dstb[vr_cell_offset(g, i, j, k)] = s_rows[((tr << rbits) + ljk) * pitch + (i - ibase)];
        }
        __syncthreads();
    }
}

/* TILED, the default 4x4x2 micro-tiles in x-fastest tile order: the same two phases with the
 * index arithmetic hoisted out of the element loops. Groups of TR = 2^TRL tile rows = 8 TR
 * source rows (TRL = 2 for small bricks, 1 when 32 rows of a large brick would take too much
 * shared memory for 6 CTAs per SM). Phase 1: warp w stages rows w, w+8, ... with cp.async (global ->
 * shared, no register stage: all of a group's 128-byte reads are in flight together); phase 2: 8/TR warps per tile row, a lane writes one 16-byte row
 * of a micro-tile (LDS.128 -> STG.128), so a warp instruction writes four whole 128-byte lines. */
__device__ __forceinline__ void cp_async4(float* smem_dst, const float* gmem_src) {
    const unsigned sa = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(sa), "l"(gmem_src) : "memory");
}

template <int TRL>
__global__ void __launch_bounds__(256)
vr_upload_tile442_kernel(VrGrid g, float* __restrict__ bricks, const float* __restrict__ src, int x0, int y0, int z0, int sx,
                         int sy, int sz, int pitch, int b0) {
    constexpr int TR = 1 << TRL;  /* tile rows per group */
    constexpr int RW = TR;        /* staged rows per warp (8 TR rows, 8 warps) */
    constexpr int CH = 8 / RW;    /* 32-cell chunks per row and iteration */
    constexpr int WPT = 8 >> TRL; /* phase 2: warps per tile row */
    extern __shared__ __align__(16) float s_rows[];
    const int b = blockIdx.y + b0; /* b0: first brick of the z range the box can touch */
    int bc[3], lo[3], hi[3];
    vr_brick_coords(g, b, bc);
    vr_brick_core(g, bc, lo, hi);
    const int ex = hi[0] - lo[0] + 2 * g.ghost, ey = hi[1] - lo[1] + 2 * g.ghost, ez = hi[2] - lo[2] + 2 * g.ghost;
    int i0, i1, j0, j1, k0, k1;
    padded_range(lo[0], g.ghost, ex, g.n[0], x0, x0 + sx, i0, i1);
    padded_range(lo[1], g.ghost, ey, g.n[1], y0, y0 + sy, j0, j1);
    padded_range(lo[2], g.ghost, ez, g.n[2], z0, z0 + sz, k0, k1);
    if (i1 <= i0 || j1 <= j0 || k1 <= k0) return;
    const int slot_b = vr_slot_index(g, b);
    if (slot_b < 0) return; /* a part handle does not hold this brick (row f3) */
    const int tx0 = i0 >> 2, tx1 = ((i1 - 1) >> 2) + 1;
    const int ty0 = j0 >> 2, ty1 = ((j1 - 1) >> 2) + 1;
    const int tz0 = k0 >> 1, tz1 = ((k1 - 1) >> 1) + 1;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int ngy = (ty1 - ty0 + TR - 1) >> TRL, groups = ngy * (tz1 - tz0);
    const int ibase = tx0 << 2;
    const int xbase = lo[0] - g.ghost; /* global x of padded cell 0 */
    const bool clamp_x = xbase < 0 || xbase + ex - 1 > g.n[0] - 1;
    float* __restrict__ dstb = bricks + (long long)slot_b * g.slot;
    /* phase-2 role of this lane: tile row tr, row r = lj + 4 lk of the tile, x tile q (+ 4 per warp of the row) */
    const int tr = warp / WPT, r = lane & 7, q = (lane >> 3) + ((warp % WPT) << 2);
    for (int grp = blockIdx.x; grp < groups; grp += gridDim.x) {
        const int tyg = ty0 + ((grp % ngy) << TRL), kt = (tz0 + grp / ngy) << 1;
        const int ntr = min(TR, ty1 - tyg);
        const float* srow[RW];
#pragma unroll
        for (int u = 0; u < RW; ++u) {
            const int rr = warp + 8 * u; /* staged row: tile row rr >> 3, lk = (rr >> 2) & 1, lj = rr & 3 */
            const int j = ((tyg + (rr >> 3)) << 2) + (rr & 3), k = kt + ((rr >> 2) & 1);
            srow[u] = NULL;
            if ((rr >> 3) < ntr && j >= j0 && j < j1 && k >= k0 && k < k1) {
                const int gy = min(max(lo[1] - g.ghost + j, 0), g.n[1] - 1), gz = min(max(lo[2] - g.ghost + k, 0), g.n[2] - 1);
                srow[u] = src + ((long long)(gz - z0) * sy + (gy - y0)) * sx + (xbase - x0);
            }
        }
        /* global -> shared without a register stage (cp.async, 4 bytes per lane): every request of the
         * group is in flight at once, whatever the compiler's scheduling; one wait before the barrier */
        for (int i = i0 + lane; i < i1; i += 32 * CH) {
#pragma unroll
            for (int c = 0; c < CH; ++c) {
                const int ic = i + 32 * c;
                if (ic < i1) {
                    const int gc = clamp_x ? min(max(xbase + ic, 0), g.n[0] - 1) - xbase : ic;
#pragma unroll
                    for (int u = 0; u < RW; ++u)
                        if (srow[u]) cp_async4(s_rows + (warp + 8 * u) * pitch + (ic - ibase), srow[u] + gc);
                }
            }
        }
        asm volatile("cp.async.commit_group;\n\tcp.async.wait_group 0;" ::: "memory");
        __syncthreads();
        {
            const int j = ((tyg + tr) << 2) + (r & 3), k = kt + (r >> 2);
            if (tr < ntr && j >= j0 && j < j1 && k >= k0 && k < k1) {
                const float* __restrict__ srw = s_rows + ((tr << 3) + r) * pitch - ibase;
                float* __restrict__ out = dstb + (vr_axis_offset(g.ax[1], j) + vr_axis_offset(g.ax[2], k));
                for (int tx = tx0 + q; tx < tx1; tx += 4 * WPT) {
                    const int i = tx << 2;
                    if (i >= i0 && i + 3 < i1) {
                        *reinterpret_cast<float4*>(out + (tx << 5)) = *reinterpret_cast<const float4*>(srw + i);
                    } else {
#pragma unroll
                        for (int c = 0; c < 4; ++c)
                            if (i + c >= i0 && i + c < i1) out[(tx << 5) + c] = srw[i + c];
                    }
                }
            }
        }
        __syncthreads();
    }
}

__global__ void __launch_bounds__(256)
vr_download_kernel(VrGrid g, const float* __restrict__ bricks, float* __restrict__ dst, int x0, int y0, int z0, int sx, int sy,
                   int sz) {
    /* one warp per row (y,z) of the requested box; lanes along x */
    const long long rows = (long long)sy * sz;
    const int warps_per_block = blockDim.x >> 5, lane = threadIdx.x & 31;
    for (long long row = (long long)blockIdx.x * warps_per_block + (threadIdx.x >> 5); row < rows;
         row += (long long)gridDim.x * warps_per_block) {
        const int y = y0 + (int)(row % sy), z = z0 + (int)(row / sy);
        const int by = y / g.brick, bz = z / g.brick;
        for (int xo = lane; xo < sx; xo += 32) {
            const int x = x0 + xo;
            const int bx = x / g.brick;
            const int b = (bz * g.g[1] + by) * g.g[0] + bx;
            const int i = x - bx * g.brick + g.ghost, j = y - by * g.brick + g.ghost, k = z - bz * g.brick + g.ghost;
            const int slot_b = vr_slot_index(g, b); /* the caller checked that the handle holds the box */
            dst[row * sx + xo] = bricks[(long long)slot_b * g.slot + vr_cell_offset(g, i, j, k)];
        }
    }
}

static cudaError_t launch_upload_tma(const VrGrid& grid, float* bricks, const float* src, int x0, int y0, int z0, int sx, int sy, int sz,
                                     int b0, unsigned nby, cudaStream_t st);
/* 1 (default) = TMA box loads (vr_upload_tma442_kernel: 5.86 TB/s on c3, 4.95 on c2) where the source allows it (sx % 4 == 0, 16-byte
 * aligned), 0 = cp.async staging (vr_upload_tile442_kernel: 5.23 / 4.83 TB/s; also the fallback) - measured round 2,
 * profiles/r2_upload.md; vr_debug_set_upload_path */
static int g_upload_path = 1;
void vr_set_upload_path(int path) { g_upload_path = path; }

cudaError_t vr_launch_upload(const VrGrid& grid, float* bricks, const float* src, int x0, int y0, int z0, int sx, int sy,
                             int sz, cudaStream_t st) {
    /* nbricks <= 65535 (checked at create): bricks along grid.y - only those brick z-slabs whose padded
     * extent can hold a plane of the box (a z-slab upload of a tall cube touches one or two of them) */
    const int bz0 = (z0 - grid.ghost) > 0 ? (z0 - grid.ghost) / grid.brick : 0;
    int bz1 = (z0 + sz - 1 + grid.ghost) / grid.brick;
    if (bz1 > grid.g[2] - 1) bz1 = grid.g[2] - 1;
    const int b0 = bz0 * grid.g[0] * grid.g[1];
    const unsigned nby = (unsigned)((bz1 - bz0 + 1) * grid.g[0] * grid.g[1]);
    if (grid.layout == VR_LAYOUT_LINEAR) {
        /* enough CTAs per brick to cover its rows once at 8 rows per CTA, capped */
        long long rows = (long long)grid.P * grid.P;
        int bx = (int)((rows + 7) / 8);
        if (bx > 4096) bx = 4096;
        vr_upload_kernel<<<dim3(bx, nby), 256, 0, st>>>(grid, bricks, src, x0, y0, z0, sx, sy, sz, b0);
    } else {
        /* one CTA per group of tile rows the box can touch in one brick, capped */
        const int rbits = grid.tl[1] + grid.tl[2];
        if (rbits > 5) return cudaErrorInvalidValue; /* a micro-tile spans at most 32 rows */
        const int TR = UP_ROWS >> rbits;
        const long long ty = (((long long)grid.P >> grid.tl[1]) + 1 + TR - 1) / TR;
        long long tz = (((long long)(sz < grid.P ? sz + 2 * grid.ghost : grid.P)) >> grid.tl[2]) + 2;
        long long bx = ty * tz;
        if (bx > 8192) bx = 8192;
        const int span = ((grid.P >> grid.tl[0]) + 1) << grid.tl[0];     /* staged cells per row */
        const int pitch = ((span + 31) / 32) * 32 + 4;                    /* = 4 (mod 32) */
        const size_t smem = sizeof(float) * (size_t)pitch * UP_ROWS;
        if (smem > 48 * 1024) {
            cudaError_t e = cudaFuncSetAttribute(vr_upload_tiled_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
            if (e != cudaSuccess) return e;
        }
        const bool t442 = grid.tl[0] == 2 && grid.tl[1] == 2 && grid.tl[2] == 1 && grid.ml[0] == 0 && grid.ml[1] == 0 &&
                          grid.ml[2] == 0;
        if (t442 && g_upload_path == 1) {
            const cudaError_t e = launch_upload_tma(grid, bricks, src, x0, y0, z0, sx, sy, sz, b0, nby, st);
            if (e != cudaErrorNotSupported) return e;
            cudaGetLastError();
        }
        if (t442) {
            /* 32 staged rows while six CTAs of them fit an SM's shared memory, else 16 */
            const bool big = smem > 40 * 1024;
            const size_t sm2 = big ? smem / 2 : smem;
            const long long ty2 = big ? (((long long)grid.P >> 2) + 2) / 2 : ty;
            long long bx2 = ty2 * tz;
            if (bx2 > 16384) bx2 = 16384;
            if (big)
                vr_upload_tile442_kernel<1><<<dim3((unsigned)bx2, nby), 256, sm2, st>>>(grid, bricks, src, x0, y0, z0, sx, sy, sz, pitch,
                                                                                        b0);
            else
                vr_upload_tile442_kernel<2><<<dim3((unsigned)bx2, nby), 256, sm2, st>>>(grid, bricks, src, x0, y0, z0, sx, sy, sz, pitch,
                                                                                        b0);
        } else {
            vr_upload_tiled_kernel<<<dim3((unsigned)bx, nby), 256, smem, st>>>(grid, bricks, src, x0, y0, z0, sx, sy, sz, pitch, b0);
        }
    }
    return cudaGetLastError();
}

cudaError_t vr_launch_download(const VrGrid& grid, const float* bricks, float* dst, int x0, int y0, int z0, int sx, int sy,
                               int sz, cudaStream_t st) {
    long long rows = (long long)sy * sz;
    long long blocks = (rows + 7) / 8;
    if (blocks > 148 * 32) blocks = 148 * 32;
    if (blocks < 1) blocks = 1;
    vr_download_kernel<<<(unsigned)blocks, 256, 0, st>>>(grid, bricks, dst, x0, y0, z0, sx, sy, sz);
    return cudaGetLastError();
}

/* ------------------------------------------------------------------------------------------
 * TILED 4x4x2, source boxes moved by the TMA unit (cp.async.bulk.tensor, sm_90+): the dense source is described by
 * a 3-D tensor map; a CTA takes a group of 4 tile rows (16 source rows x 2 planes) of one brick and walks it in
 * chunks of 128 cells: one elected thread asks for the next chunk's 132 x 16 x 2 box (16.5 KB, out-of-range
 * coordinates are filled with zeros by the unit and never used) while all threads turn the previous chunk into
 * micro-tiles, two shared-memory stages, one mbarrier each. Against the cp.async version: no address arithmetic and no
 * 4-byte requests on the load side - but the unit wants every box to start on a 16-byte boundary of the source row
 * (a box at x = -1 faults as an illegal instruction), so with one ghost layer the staged rows sit 3 cells askew: a
 * 16-byte tile row is picked out of TWO aligned 128-bit shared loads. First version (four 4-byte shared loads per row,
 * a warp store over eight half-lines): 5 % slower than the cp.async kernel on c3. With whole-line stores and aligned
 * conflict-free loads (the lane mapping in the kernel), the per-unit tests hoisted and a narrow box for a row's ghost-cell tail:
 * 35.41 against 39.65 ms for c3's 207 GB (5.86 against 5.23 TB/s), 1.754 against 1.799 ms on c2 - the default. Three or four stages (fewer CTAs per SM) and 8-row boxes are slower
 * (profiles/r2_upload.md). Needs sx % 4 == 0 and a 16-byte aligned source (the tensor map's strides), else the caller
 * falls back to the cp.async kernel.
 * ---------------------------------------------------------------------------------------- */
#include <cuda.h>

#define TMA_BX 128 /* cells per chunk */
#define TMA_BW (TMA_BX + 4) /* box width: the unit wants the box to start on a 16-byte boundary of the source row, so it starts
                             * up to 3 cells early (a ghost layer of 1 puts padded cell 0 at voxel -1 mod 4) */
#ifndef TMA_TR
#define TMA_TR 4   /* tile rows per group: 16 source rows */
#endif
#define TMA_STAGE_FLOATS (TMA_BW * TMA_TR * 4 * 2)
#define TMA_TW 8    /* box width of a brick row's TAIL: the last chunk of a 128 k + 2 ghost cells wide row holds 2 or 4 cells (+ up to 3 of skew);
                     * a full-width box there would read 132 cells for them (c3: 660 cells read per row of 514) */
#ifndef VR_TMA_STAGES
#define VR_TMA_STAGES 2 /* shared-memory stages (boxes in flight per CTA) */
#endif

__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long* bar, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long* bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long* bar, unsigned parity) {
    unsigned done = 0;
    while (!done)
        asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                     : "=r"(done)
                     : "r"(smem_u32(bar)), "r"(parity)
                     : "memory");
}
__device__ __forceinline__ void tma_load_3d(float* dst, const CUtensorMap* tm, unsigned long long* bar, int x, int y, int z) {
    asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];" ::"r"(
                     smem_u32(dst)),
                 "l"(tm), "r"(smem_u32(bar)), "r"(x), "r"(y), "r"(z)
                 : "memory");
}

__global__ void __launch_bounds__(256)
vr_upload_tma442_kernel(VrGrid g, float* __restrict__ bricks, const __grid_constant__ CUtensorMap tm, const __grid_constant__ CUtensorMap tm_tail,
                        const float* __restrict__ src,
                        int x0, int y0, int z0, int sx, int sy, int sz, int b0) {
    extern __shared__ __align__(128) float s_box_raw[]; /* two stages of [2][16][128] floats, 128-byte aligned by hand */
    __shared__ __align__(8) unsigned long long s_bar[VR_TMA_STAGES];
    float* s_box = reinterpret_cast<float*>((reinterpret_cast<uintptr_t>(s_box_raw) + 127) & ~(uintptr_t)127);
    const int b = blockIdx.y + b0;
    int bc[3], lo[3], hi[3];
    vr_brick_coords(g, b, bc);
    vr_brick_core(g, bc, lo, hi);
    const int ex = hi[0] - lo[0] + 2 * g.ghost, ey = hi[1] - lo[1] + 2 * g.ghost, ez = hi[2] - lo[2] + 2 * g.ghost;
    int i0, i1, j0, j1, k0, k1;
    padded_range(lo[0], g.ghost, ex, g.n[0], x0, x0 + sx, i0, i1);
    padded_range(lo[1], g.ghost, ey, g.n[1], y0, y0 + sy, j0, j1);
    padded_range(lo[2], g.ghost, ez, g.n[2], z0, z0 + sz, k0, k1);
    if (i1 <= i0 || j1 <= j0 || k1 <= k0) return;
    const int slot_b = vr_slot_index(g, b);
    if (slot_b < 0) return;
    const int tx0 = i0 >> 2, tx1 = ((i1 - 1) >> 2) + 1;
    const int ty0 = j0 >> 2, ty1 = ((j1 - 1) >> 2) + 1;
    const int tz0 = k0 >> 1, tz1 = ((k1 - 1) >> 1) + 1;
    const int ngy = (ty1 - ty0 + TMA_TR - 1) / TMA_TR, groups = ngy * (tz1 - tz0);
    const int xbase = lo[0] - g.ghost, ybase = lo[1] - g.ghost, zbase = lo[2] - g.ghost; /* global voxel of padded cell 0 */
    float* __restrict__ dstb = bricks + (long long)slot_b * g.slot;
    const int xskew = (xbase + (tx0 << 2) - x0) & 3; /* cells between the box's 16-byte aligned start and the chunk's first cell */
    /* chunks of 128 cells; a last chunk of a few cells (the ghost layers of a 128 k wide brick) comes in a narrow box. (Letting it ride
     * along with the last full chunk in a 140-cell box - one unit less per group - was 14 % slower: profiles/r2_upload.md) */
    const int nchunks = (i1 - (tx0 << 2) + TMA_BX - 1) / TMA_BX;
    const int tid = threadIdx.x;
    /* phase-2 role of this thread (see the loop): row lj of plane lk of the tile txl of a chunk */
    const int lane_lj = tid & 3, lane_lk = (tid >> 3) & 1;
    const int lane_txl = ((tid >> 5) & 3) | (((tid >> 2) & 1) << 2) | (((tid >> 4) & 1) << 3) | (((tid >> 7) & 1) << 4);
    if (tid == 0) {
        for (int q = 0; q < VR_TMA_STAGES; ++q) mbar_init(&s_bar[q], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    /* work units of this CTA: (group, chunk), group = blockIdx.x, blockIdx.x + gridDim.x, ... */
    const int my_groups = groups > (int)blockIdx.x ? (groups - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x : 0;
    const int units = my_groups * nchunks;
    auto issue = [&](int u) {
        const int grp = (int)blockIdx.x + (u / nchunks) * (int)gridDim.x, c = u % nchunks;
        const int jf = (ty0 + (grp % ngy) * TMA_TR) << 2, kt = (tz0 + grp / ngy) << 1, ic = (tx0 << 2) + c * TMA_BX;
        unsigned long long* bar = &s_bar[u % VR_TMA_STAGES];
        const bool tail = (i1 - ic) + xskew <= TMA_TW; /* the narrow box holds everything this chunk needs */
        mbar_expect_tx(bar, (tail ? TMA_TW : TMA_BW) * (TMA_TR * 4 * 2) * 4u);
        tma_load_3d(s_box + (u % VR_TMA_STAGES) * TMA_STAGE_FLOATS, tail ? &tm_tail : &tm, bar, (xbase + ic - x0) & ~3, ybase + jf - y0,
                    zbase + kt - z0);
    };
    if (tid == 0)
        for (int u = 0; u < VR_TMA_STAGES - 1 && u < units; ++u) issue(u);
    for (int u = 0; u < units; ++u) {
        if (tid == 0 && u + VR_TMA_STAGES - 1 < units) issue(u + VR_TMA_STAGES - 1); /* its stage was released by the barrier that ended unit u - 1 */
        mbar_wait(&s_bar[u % VR_TMA_STAGES], (unsigned)((u / VR_TMA_STAGES) & 1));
        const int grp = (int)blockIdx.x + (u / nchunks) * (int)gridDim.x, c = u % nchunks;
        const int tyg = ty0 + (grp % ngy) * TMA_TR, kt = (tz0 + grp / ngy) << 1, ic = (tx0 << 2) + c * TMA_BX;
        const float* __restrict__ box = s_box + (u % VR_TMA_STAGES) * TMA_STAGE_FLOATS;
        /* 1024 sixteen-byte tile rows per unit (TMA_TR = 4), 4 per thread. A warp takes the 8 rows (lj, lk) of FOUR tiles, so its store
         * covers four whole 128-byte lines; a quarter-warp (one 128-bit shared-load wavefront) takes the rows lj = 0..3 of one
         * plane lk of the tiles t and t + 4: rows are 132 floats apart (4 banks), tiles 4 floats, so its eight 16-byte words
         * fall into eight different bank groups - also one word further on (the second load of an askew row) */
        /* idx = tid + 256 n: a thread keeps its row (lj, lk) and its tile txl (lane_* above) in every round; n is the tile row.
         * What does not depend on n is tested once per unit. */
        const int pitch = (i1 - ic) + xskew <= TMA_TW ? TMA_TW : TMA_BW; /* as issued */
        const int txl = lane_txl;
        const int tx = (ic >> 2) + txl, i = tx << 2, k = kt + lane_lk;
        if (tx < tx1 && k >= k0 && k < k1) {
            const int gz = zbase + k, gx = xbase + i;
            /* cells outside the volume replicate the edge voxel (R3): the unit filled them with zeros, so the few rows and
             * columns on the volume's faces take the clamped voxel straight from the source (it lies in the box: padded_range) */
            const bool edge_xz = gz < 0 || gz >= g.n[2] || gx < 0 || gx + 3 >= g.n[0];
            const bool whole = i >= i0 && i + 3 < i1;
            const float* __restrict__ scol = box + (lane_lk * (TMA_TR * 4) + lane_lj) * pitch + (txl << 2);
            float* __restrict__ ocol = dstb + vr_axis_offset(g.ax[2], k) + (tx << 5);
#pragma unroll
            for (int n = 0; n < TMA_TR; ++n) { /* 256 TMA_TR tile rows per unit */
                const int j = ((tyg + n) << 2) + lane_lj;
                if (tyg + n >= ty1 || j < j0 || j >= j1) continue;
                const float* __restrict__ srow = scol + n * (4 * pitch); /* 16-byte aligned; the cells start xskew further on */
                float* __restrict__ out = ocol + vr_axis_offset(g.ax[1], j);
                const int gy = ybase + j;
                const bool edge = edge_xz || gy < 0 || gy >= g.n[1];
                if (!edge && whole) {
                    /* an askew row: two aligned 128-bit loads and a pick (xskew is the same for the whole CTA) */
                    const float4 A = *reinterpret_cast<const float4*>(srow);
                    float4 v = A;
                    if (xskew) {
                        const float4 B = *reinterpret_cast<const float4*>(srow + 4);
                        v = xskew == 1 ? make_float4(A.y, A.z, A.w, B.x) : xskew == 2 ? make_float4(A.z, A.w, B.x, B.y) : make_float4(A.w, B.x, B.y, B.z);
                    }
                    *reinterpret_cast<float4*>(out) = v;
                } else if (!edge) {
#pragma unroll
                    for (int q = 0; q < 4; ++q)
                        if (i + q >= i0 && i + q < i1) out[q] = srow[xskew + q];
                } else {
                    const int cy = min(max(gy, 0), g.n[1] - 1), cz = min(max(gz, 0), g.n[2] - 1);
                    const float* __restrict__ grow = src + ((long long)(cz - z0) * sy + (cy - y0)) * sx - x0;
#pragma unroll
                    for (int q = 0; q < 4; ++q)
                        if (i + q >= i0 && i + q < i1) out[q] = __ldg(grow + min(max(gx + q, 0), g.n[0] - 1));
                }
            }
        }
        __syncthreads();
    }
}

typedef CUresult (*vr_encode_tiled_fn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                       const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                       CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

/* Returns cudaErrorNotSupported when the source cannot be described by a tensor map (or the driver has no encoder): the
 * caller then falls back to the cp.async kernel. */
static cudaError_t launch_upload_tma(const VrGrid& grid, float* bricks, const float* src, int x0, int y0, int z0, int sx, int sy, int sz,
                                     int b0, unsigned nby, cudaStream_t st) {
    static vr_encode_tiled_fn encode = NULL;
    static bool looked = false;
    if (!looked) {
        looked = true;
        void* fn = NULL;
        cudaDriverEntryPointQueryResult qr;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qr) == cudaSuccess && qr == cudaDriverEntryPointSuccess)
            encode = (vr_encode_tiled_fn)fn;
        cudaGetLastError();
    }
    if (!encode || (sx & 3) || (((uintptr_t)src) & 15)) return cudaErrorNotSupported;
    CUtensorMap tm;
    const cuuint64_t dims[3] = {(cuuint64_t)sx, (cuuint64_t)sy, (cuuint64_t)sz};
    const cuuint64_t strides[2] = {(cuuint64_t)sx * 4, (cuuint64_t)sx * sy * 4};
    const cuuint32_t box[3] = {TMA_BW, TMA_TR * 4, 2};
    const cuuint32_t estr[3] = {1, 1, 1};
    if (encode(&tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, (void*)src, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
               CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
        return cudaErrorNotSupported;
    CUtensorMap tm_tail;
    const cuuint32_t box_tail[3] = {TMA_TW, TMA_TR * 4, 2};
    if (encode(&tm_tail, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, (void*)src, dims, strides, box_tail, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
               CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
        return cudaErrorNotSupported;
    const size_t smem = VR_TMA_STAGES * TMA_STAGE_FLOATS * sizeof(float) + 128;
    cudaError_t e = cudaFuncSetAttribute(vr_upload_tma442_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    const long long ty = (((long long)grid.P >> 2) + 1 + TMA_TR - 1) / TMA_TR;
    const long long tz = (((long long)(sz < grid.P ? sz + 2 * grid.ghost : grid.P)) >> 1) + 2;
    long long bx = ty * tz;
    if (bx > 4096) bx = 4096;
    vr_upload_tma442_kernel<<<dim3((unsigned)bx, nby), 256, smem, st>>>(grid, bricks, tm, tm_tail, src, x0, y0, z0, sx, sy, sz, b0);
    return cudaGetLastError();
}
