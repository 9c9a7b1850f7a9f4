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
 * writes, coalesced reads except at the two replicated ends). TILED: one warp per micro-tile
 * (one coalesced 128-byte line written; the 16-byte source segments it reads are shared with
 * the neighbouring warps of the CTA through L1). A cell is written iff its clamped global
 * index lies in the uploaded box, which makes z-slab uploads of a ~100 GB cube work.
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
                 int sz) {
    const int b = blockIdx.y;
    int bc[3], lo[3], hi[3];
    vr_brick_coords(g, b, bc);
    vr_brick_core(g, bc, lo, hi);
    const int ex = hi[0] - lo[0] + 2 * g.ghost, ey = hi[1] - lo[1] + 2 * g.ghost, ez = hi[2] - lo[2] + 2 * g.ghost;
    int i0, i1, j0, j1, k0, k1;
    padded_range(lo[0], g.ghost, ex, g.n[0], x0, x0 + sx, i0, i1);
    padded_range(lo[1], g.ghost, ey, g.n[1], y0, y0 + sy, j0, j1);
    padded_range(lo[2], g.ghost, ez, g.n[2], z0, z0 + sz, k0, k1);
    if (i1 <= i0 || j1 <= j0 || k1 <= k0) return;
    const int rows = (j1 - j0) * (k1 - k0);
    const int warps_per_block = blockDim.x >> 5, lane = threadIdx.x & 31;
    float* __restrict__ dstb = bricks + (long long)b * g.slot;
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

/* TILED: CTA = one row of micro-tiles (fixed tile y, z) of one brick; warp w takes tiles
 * w, w+8, ... along x; lane = cell inside the tile. */
__global__ void __launch_bounds__(256)
vr_upload_tiled_kernel(VrGrid g, float* __restrict__ bricks, const float* __restrict__ src, int x0, int y0, int z0, int sx,
                       int sy, int sz) {
    const int b = blockIdx.y;
    int bc[3], lo[3], hi[3];
    vr_brick_coords(g, b, bc);
    vr_brick_core(g, bc, lo, hi);
    const int ex = hi[0] - lo[0] + 2 * g.ghost, ey = hi[1] - lo[1] + 2 * g.ghost, ez = hi[2] - lo[2] + 2 * g.ghost;
    int i0, i1, j0, j1, k0, k1;
    padded_range(lo[0], g.ghost, ex, g.n[0], x0, x0 + sx, i0, i1);
    padded_range(lo[1], g.ghost, ey, g.n[1], y0, y0 + sy, j0, j1);
    padded_range(lo[2], g.ghost, ez, g.n[2], z0, z0 + sz, k0, k1);
    if (i1 <= i0 || j1 <= j0 || k1 <= k0) return;
    const int tx0 = i0 >> g.tl[0], tx1 = ((i1 - 1) >> g.tl[0]) + 1;
    const int ty0 = j0 >> g.tl[1], ty1 = ((j1 - 1) >> g.tl[1]) + 1;
    const int tz0 = k0 >> g.tl[2], tz1 = ((k1 - 1) >> g.tl[2]) + 1;
    const int rows = (ty1 - ty0) * (tz1 - tz0);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, nwarps = blockDim.x >> 5;
    const int li = lane & ((1 << g.tl[0]) - 1), lj = (lane >> g.tl[0]) & ((1 << g.tl[1]) - 1), lk = lane >> (g.tl[0] + g.tl[1]);
    float* __restrict__ dstb = bricks + (long long)b * g.slot;
    for (int row = blockIdx.x; row < rows; row += gridDim.x) {
        const int j = ((ty0 + row % (ty1 - ty0)) << g.tl[1]) + lj, k = ((tz0 + row / (ty1 - ty0)) << g.tl[2]) + lk;
        if (j < j0 || j >= j1 || k < k0 || k >= k1) continue;
        const int gy = min(max(lo[1] - g.ghost + j, 0), g.n[1] - 1), gz = min(max(lo[2] - g.ghost + k, 0), g.n[2] - 1);
        const float* __restrict__ srow = src + ((long long)(gz - z0) * sy + (gy - y0)) * sx;
        const unsigned oyz = vr_axis_offset(g.ax[1], j) + vr_axis_offset(g.ax[2], k);
        for (int t = tx0 + warp; t < tx1; t += nwarps) {
            const int i = (t << g.tl[0]) + li;
            if (i < i0 || i >= i1) continue;
            const int gx = min(max(lo[0] - g.ghost + i, 0), g.n[0] - 1);
            dstb[oyz + vr_axis_offset(g.ax[0], i)] = __ldg(srow + (gx - x0));
        }
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
            dst[row * sx + xo] = bricks[(long long)b * g.slot + vr_cell_offset(g, i, j, k)];
        }
    }
}

cudaError_t vr_launch_upload(const VrGrid& grid, float* bricks, const float* src, int x0, int y0, int z0, int sx, int sy,
                             int sz, cudaStream_t st) {
    /* nbricks <= 65535 (checked at create): bricks along grid.y */
    if (grid.layout == VR_LAYOUT_LINEAR) {
        /* enough CTAs per brick to cover its rows once at 8 rows per CTA, capped */
        long long rows = (long long)grid.P * grid.P;
        int bx = (int)((rows + 7) / 8);
        if (bx > 4096) bx = 4096;
        vr_upload_kernel<<<dim3(bx, grid.nbricks), 256, 0, st>>>(grid, bricks, src, x0, y0, z0, sx, sy, sz);
    } else {
        /* one CTA per row of micro-tiles the box can touch in one brick, capped */
        const long long ty = ((long long)grid.P >> grid.tl[1]) + 1;
        long long tz = (((long long)(sz < grid.P ? sz + 2 * grid.ghost : grid.P)) >> grid.tl[2]) + 2;
        long long bx = ty * tz;
        if (bx > 8192) bx = 8192;
        vr_upload_tiled_kernel<<<dim3((unsigned)bx, grid.nbricks), 256, 0, st>>>(grid, bricks, src, x0, y0, z0, sx, sy, sz);
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
