/*
 * vr_internal.cuh -- shared declarations of libvr's translation units (not part of the ABI).
 *
 * Data layout in HBM:
 *   bricks        float[nown][slot], P = brick + 2*ghost padded cells per axis. Brick b =
 *                 (bz*gy + by)*gx + bx sits in slot vr_slot_index(b) (= b unless the handle is a part). Padded cell (i,j,k) of brick b holds global voxel
 *                 clamp(lo_b - ghost + (i,j,k), 0, n-1) and sits at vr_cell_offset(i,j,k):
 *                 x-linear rows (VR_LAYOUT_LINEAR) or 128-byte 3-D micro-tiles
 *                 (VR_LAYOUT_TILED), see VrAxisLayout. Ragged bricks use the low corner of
 *                 their slot. 64-bit offsets throughout (a 104 GB store has 2.6e10 cells).
 *   VrViewState   one per handle: matrices, eye, totals, work counter (written by set-up).
 *   VrBrickView   one per brick: rendering rectangle, launch rectangle, sub-image offset.
 *   order         int[nbricks]: brick ids front to back; item_prefix int[nbricks+1]:
 *                 exclusive prefix of work-item counts by order position.
 *   sub-images    per brick, launch-rectangle sized, float4 (ALPHA) or float (MIP) per pixel.
 */
#ifndef VR_INTERNAL_CUH
#define VR_INTERNAL_CUH

#include <cuda_runtime.h>
#include <stddef.h>
#include <stdint.h>

#include "../../include/vr.h"

#define VR_MAX_LUT 1024
#define VR_TILE_W 8 /* a warp renders an 8x4 pixel tile of one brick */
#define VR_TILE_H 4
#define VR_MAX_AXIS_BRICKS 1024
#define VR_RAYCAST_THREADS 256
#define VR_COMP_TILE_W 32
#define VR_COMP_TILE_H 8
/* internal compositing modes next to VR_ALPHA / VR_MIP (row f3):
 *   VR_MIP_RAW    scalar MIP sub-images in, scalar maximum out (-inf where no layer holds a sample)
 *   VR_MIP_PARTS  such scalar partial frames in, LUT colour of the maximum out ((0,0,0,0) where all are -inf) */
#define VR_MIP_RAW 2
#define VR_MIP_PARTS 3
#define VR_EV_RING 64 /* timed frames whose stage events are kept */

/* Where padded cell i of one axis sits inside a brick slot. Every supported layout is
 * SEPARABLE: offset(i,j,k) = ax[0](i) + ax[1](j) + ax[2](k) floats, with
 *   ax(i) = ((i & lo_mask) << lo_shift)                        position inside a 128-byte micro-tile
 *         + (((i >> mid_in) & mid_mask) << mid_shift)          micro-tile inside a macro block
 *         + (i >> hi_in) * hi_stride                           macro block (or tile) along this axis
 * x-linear rows are the special case lo_mask = ~0 (x) / hi_in = 0, hi_stride = P, P*P (y, z). */
struct VrAxisLayout {
    int lo_mask, lo_shift;
    int mid_in, mid_mask, mid_shift;
    int hi_in;
    unsigned hi_stride;
};

struct VrGrid {
    int n[3];     /* nx, ny, nz */
    int g[3];     /* bricks per axis */
    int brick, ghost;
    int nbricks;
    int P;        /* padded edge of a brick slot */
    long long slot; /* floats per brick slot (a multiple of 32: slots start on 128-byte lines) */
    int brick_pow2; /* 1 if brick is a power of two (division by it is an exact scaling) */
    int layout;     /* VR_LAYOUT_LINEAR or VR_LAYOUT_TILED */
    int tl[3];      /* log2 edge of a micro-tile (tiled: 2^(tl0+tl1+tl2) = 32 floats = 128 bytes) */
    int ml[3];      /* log2 micro-tiles per macro block and axis (0,0,0: tiles in x-fastest order) */
    int nt[3];      /* tiled: macro blocks (or tiles) per axis of a slot */
    VrAxisLayout ax[3];
    /* row f3: a PART handle stores only the bricks of the box pb0 <= (bx,by,bz) < pb1 of the global grid, in
     * box-local x-fastest order (slot index, vr_slot_index); a whole volume has the box of the whole grid */
    int part;       /* 1 if the box is smaller than the grid */
    int pb0[3], pb1[3];
    int nown;       /* bricks in the box = slots of the store and rows of the macro-cell tables */
};

/* The caller's matrices travel to the set-up kernel as a kernel argument (no copy, no sync). */
struct VrMatrices {
    float view[16];
    float proj[16];
};

struct VrViewState {
    double M[16];    /* proj * view, column-major */
    double Minv[16];
    double eye[3];   /* perspective: eye point; orthographic: forward direction (R9) */
    int ortho;
    int singular;
    int W, H;
    int total_items;
    int overflow;
    long long total_sub_pixels;
    unsigned int work_counter;
    unsigned int pad0;
    unsigned long long samples;
    float data_max; /* global maximum of the data if known, else +inf (MIP stop) */
    int culled;     /* bricks skipped as transparent in this view (R16) */
    int bound[4];   /* union of the non-empty rendering rectangles (x0, y0, x1, y1; zeros if none): the frame is
                     * blank outside it, which the compositing kernel uses to leave early */
};

static_assert(offsetof(VrViewState, bound) % 16 == 0, "VrViewState::bound is read as one int4");

struct VrBrickView {
    int rx0, ry0, rx1, ry1; /* rendering rectangle, half-open, clipped */
    int lx0, ly0, lx1, ly1; /* launch rectangle: the same, grown to the 8x4 tile grid */
    int tiles_x, tiles_y;
    int order_pos;
    int slot;               /* vr_slot_index of the brick (-1: held by another part) */
    long long sub_offset;   /* first pixel of this brick's sub-image in the scratch */
};

/* One layer of the sort-last compositing pass (a brick sub-image or a caller's layer). */
struct VrCompLayer {
    int x0, y0, x1, y1;      /* pixels of the frame this layer covers (half-open) */
    int sx0, sy0;            /* frame position of the layer's stored pixel (0,0) */
    int pitch;               /* stored pixels per row */
    int pad;
    unsigned long long addr; /* device address of stored pixel (0,0) */
};

struct VrLut {
    const float4* base;  /* device: entries LUT[i]           (n of them)   */
    const float4* delta; /* device: LUT[i+1] - LUT[i]         (n-1, last 0) */
    int n;
    float vmin, vmax, inv_range;
    int nm2;     /* n - 2: last interval */
    float scale; /* n - 1 as float: u -> table coordinate */
};

/* Per-frame ray table ("each GPU kernel then starts by calculating its ray's start location,
 * orientation" - once per RAY, not once per (ray, brick)). Planes of W*H entries, entry of pixel (i, j) at j*W + i:
 *   four double2 planes  (o0, o1) (o2, d0) (d1, d2) (t0, t1)                                 64 bytes per pixel
 *   one int plane        K, the number of scheduled samples (0 = the ray misses the volume)    4
 *   one double plane     the ray's step, written only for VR_STEP_AUTO (R18)                   8
 * = VR_RAY_BYTES per pixel of scratch. Written by vr_rays_kernel for the pixels inside VrViewState::bound,
 * read by the ray-cast kernel (64 to 76 bytes per (ray, brick) segment). */
#define VR_RAY_BYTES 80 /* 76 rounded up: the planes stay 16-byte aligned for any W*H */

struct VrRaycastParams {
    VrGrid grid;
    const float* bricks;
    const double2* rays; /* the frame's ray table */
    long long ray_plane; /* entries per plane = W*H */
    const VrViewState* vs;
    const VrBrickView* bv;
    const int* order;
    const int* item_prefix;
    VrViewState* vs_rw; /* work counter, sample counter */
    void* sub;          /* float4[] (ALPHA) or float[] (MIP) */
    const cudaTextureObject_t* tex; /* texture arm (vr_texture.cu): one texture object per slot, or NULL = hand-rolled sampling */
    const int* tex_nan;             /* 1 per slot that holds blanked voxels: sampled by hand also in the texture arm (R14) */
    const float2* brick_mm;         /* texture arm, MIP: (min, max) of every brick's padded cells (row f1), indexed by brick */
    float mip_range_eps;            /* texture arm, MIP: the filter's error bound as a fraction of the brick's range (1/64; byte texels + 1/500) */
    float mip_mag_eps;              /* ... and the part that scales with the magnitude (2^-14; float16 texels 2^-9; byte texels 2^-12) */
    float mip_abs_eps;              /* ... and the absolute part: float16 texels are 2^-24 apart below 2^-14 (subnormals), rounded twice */
    int tex_byte;                   /* byte texels: a fetch returns (v - min) / (max - min) of the brick */
    float mip_mag_max;              /* bricks with a larger magnitude keep the hand-rolled loop (float16 texels: 60000; else inf) */
    unsigned* bitmap;   /* counting variant only: one bit per brick-store cell, or NULL */
    const unsigned* cell_bits; /* R19: one bit per 8x8x8 macro-cell, 1 = transparent under the LUT; NULL = no skipping */
    const float2* cell_mm; /* R19, MIP: (min, max) per macro-cell (a cell whose max cannot raise the ray's maximum is skipped); NULL = off */
    int nc[3];          /* macro-cells per axis of a brick slot */
    int cell_words;     /* 32-bit words of cell_bits per brick */
    VrLut lut;
    int lut_copies; /* copies of the table in the ray-cast kernel's shared memory (vr_lut_copies) */
    float tex_guard; /* texture arm, ALPHA, steps below one voxel: a sample whose table opacity exceeds this is evaluated by the hand-rolled
                      * sampler instead (the opacity correction (1 - a)^w has an unbounded slope at a = 1 for w < 1: R20); > 1 = off */
    int tex_only;    /* the float32 store was released: the exit samples go through the arrays too */
    double step; /* > 0: sample spacing in voxels; 0: per ray, 1 / max|d_a| (R18) */
    float tau;
    int mode;
};

/* Offset (floats) of padded cell (i,j,k) inside a brick slot; < 2^32 for every legal slot. */
__host__ __device__ __forceinline__ unsigned vr_axis_offset(const VrAxisLayout& A, int i) {
    return ((unsigned)(i & A.lo_mask) << A.lo_shift) + ((unsigned)((i >> A.mid_in) & A.mid_mask) << A.mid_shift) +
           (unsigned)(i >> A.hi_in) * A.hi_stride;
}
__host__ __device__ __forceinline__ int vr_slot_of_coords(const VrGrid& g, const int bc[3]) {
    if (!g.part) return (bc[2] * g.g[1] + bc[1]) * g.g[0] + bc[0];
    if (bc[0] < g.pb0[0] || bc[0] >= g.pb1[0] || bc[1] < g.pb0[1] || bc[1] >= g.pb1[1] || bc[2] < g.pb0[2] || bc[2] >= g.pb1[2]) return -1;
    return ((bc[2] - g.pb0[2]) * (g.pb1[1] - g.pb0[1]) + (bc[1] - g.pb0[1])) * (g.pb1[0] - g.pb0[0]) + (bc[0] - g.pb0[0]);
}
/* Slot of brick b in this handle's store (b itself for a whole volume), -1 if the handle does not hold it. */
__host__ __device__ __forceinline__ int vr_slot_index(const VrGrid& g, int b) {
    if (!g.part) return b;
    const int t = b / g.g[0];
    const int bx = b - t * g.g[0], bz = t / g.g[1], by = t - bz * g.g[1];
    if (bx < g.pb0[0] || bx >= g.pb1[0] || by < g.pb0[1] || by >= g.pb1[1] || bz < g.pb0[2] || bz >= g.pb1[2]) return -1;
    return ((bz - g.pb0[2]) * (g.pb1[1] - g.pb0[1]) + (by - g.pb0[1])) * (g.pb1[0] - g.pb0[0]) + (bx - g.pb0[0]);
}
__host__ __device__ __forceinline__ unsigned vr_cell_offset(const VrGrid& g, int i, int j, int k) {
    return vr_axis_offset(g.ax[0], i) + vr_axis_offset(g.ax[1], j) + vr_axis_offset(g.ax[2], k);
}

/* ---- launchers (each returns the cudaError of its launch) ---- */
/* range: float2[nbricks + 1] (per brick, then the whole volume) or NULL = unknown, no culling */
cudaError_t vr_launch_setup(const VrGrid& grid, const VrMatrices& mats, int W, int H, int mode,
                            long long sub_capacity_px, void* sub_base, VrViewState* vs, VrBrickView* bv, int* order,
                            int* item_prefix, VrCompLayer* layers, const float2* range, const VrLut& lut, int* overflow_flag,
                            cudaStream_t st);
/* texture arm of the brick store (vr_texture.cu): one 3-D CUDA array + texture object per slot */
struct VrTexStore;
#define VR_TEXEL_FLOAT 0
#define VR_TEXEL_HALF 1
#define VR_TEXEL_BYTE 2
cudaError_t vr_tex_create(const VrGrid& grid, VrTexStore** out, bool all, int texel);
cudaError_t vr_tex_convert_slot(const VrGrid& grid, const float* bricks, VrTexStore* t, int s, int* has_nan, cudaStream_t st);
/* a store that can be handed back slot by slot (vr_vmm.cu: CUDA virtual memory management) */
struct VrVmm;
cudaError_t vr_vmm_create(size_t slot_bytes, int nslots, VrVmm** out, float** base_out);
void vr_vmm_destroy(VrVmm* m);
size_t vr_vmm_release_slot(VrVmm* m, int s);
int vr_vmm_slot_released(const VrVmm* m, int s);
void vr_tex_destroy(VrTexStore* t);
const cudaTextureObject_t* vr_tex_table(const VrTexStore* t);
const int* vr_tex_nan_table(const VrTexStore* t);
int vr_tex_texel(const VrTexStore* t);
cudaError_t vr_launch_tex_error(const VrGrid& grid, const float* bricks, const VrTexStore* t, int s, long long n, unsigned seed, float dec_a,
                                float dec_b, float* max_err, cudaStream_t st);
cudaError_t vr_launch_tex_fill(const VrGrid& grid, const float* bricks, const VrTexStore* t, const float2* brick_mm, cudaStream_t st);
/* ray table of the frame whose set-up is in vs (row a4, the per-ray part) */
cudaError_t vr_launch_rays(const VrGrid& grid, const VrViewState* vs, int W, int H, double step, double2* rays, cudaStream_t st);
cudaError_t vr_launch_minmax(const VrGrid& grid, const float* bricks, int2* enc, float2* table, cudaStream_t st);
/* rows f1 + R19 in one streaming read (4x4x2 layout, ghost >= 1): the per-brick table and the macro-cell table; 4 launches */
/* slot_ext: device int4[nown], the padded extent (x, y, z) of the brick in each slot */
cudaError_t vr_launch_ranges(const VrGrid& grid, const float* bricks, int2* enc, float2* table, float2* cell_mm, const int nc[3],
                             const int4* slot_ext, cudaStream_t st);
/* macro-cells (R19): per-cell (min, max) of the 4x4x2-tiled store; transparency bits for a LUT */
cudaError_t vr_launch_cell_minmax(const VrGrid& grid, const float* bricks, float2* cell_mm, const int nc[3], cudaStream_t st);
/* *count += macro-cells of the whole store whose (min, max) is exactly (lo, lo): empty space of a density cube */
cudaError_t vr_launch_cell_range_sum(const float2* cell_mm, long long ncells, double* stat, cudaStream_t st);
cudaError_t vr_launch_cell_count_empty(const float2* cell_mm, long long ncells, const float2* global_mm, unsigned long long* count,
                                       cudaStream_t st);
cudaError_t vr_launch_cell_flags(const float2* cell_mm, unsigned* bits, int nbricks, const int nc[3], int words_per_brick,
                                 const VrLut& lut, cudaStream_t st);
/* items = work items of the view (sizes the persistent grid); sparse = the view samples the store at
 * more than two voxels per pixel (launch heuristic only) */
cudaError_t vr_launch_raycast(const VrRaycastParams& p, long long items, bool count, bool sparse, cudaStream_t st);
/* fused traversal (row f2): one ray per frame pixel through all bricks, writes the frame */
cudaError_t vr_launch_fused(const VrRaycastParams& p, float* frame, int W, int H, bool count, cudaStream_t st);
/* bound: device int[4] as VrViewState::bound, or NULL (layers anywhere); window: host int[4] (x0, y0, x1, y1), the
 * pixels of the W x H frame this launch writes, stored [y1-y0][x1-x0] at out, or NULL = the whole frame.
 * out: float4 per pixel, except VR_MIP_RAW: one float per pixel (-inf = no sample). */
cudaError_t vr_launch_composite(const VrCompLayer* layers, const int* order, int n, int W, int H, int mode,
                                const VrLut& lut, float* out, const int* bound, const int* window, cudaStream_t st);
cudaError_t vr_launch_upload(const VrGrid& grid, float* bricks, const float* src, int x0, int y0, int z0, int sx,
                             int sy, int sz, cudaStream_t st);
void vr_set_upload_path(int path); /* 0 cp.async staging, 1 TMA box loads (default where it applies) */
cudaError_t vr_launch_download(const VrGrid& grid, const float* bricks, float* dst, int x0, int y0, int z0, int sx,
                               int sy, int sz, cudaStream_t st);
cudaError_t vr_launch_ray_bricks(const VrGrid& grid, const VrViewState* vs, const int* d_pixels, int npix,
                                 int* d_counts, int* d_lists, double* d_tins, int maxlen, unsigned char* d_grazing,
                                 cudaStream_t st);
cudaError_t vr_launch_gather_sub(const VrBrickView* bv, int nbricks, const void* sub, int mode, const int* d_pixels,
                                 int npix, float* d_out, cudaStream_t st);
cudaError_t vr_launch_brick_copy(const VrGrid& grid, const float* bricks, int b, const int dims[3], float* d_out,
                                 cudaStream_t st);
cudaError_t vr_launch_count_bits(const unsigned* bitmap, long long words, unsigned long long* d_out3, cudaStream_t st);

/* host mirror of the set-up arithmetic, for argument validation and scratch sizing only */
int vr_host_view_check(const VrGrid& grid, const float* view, const float* proj, int W, int H, long long* sub_pixels,
                       long long* items);

int vr_host_part_rect(const VrGrid& grid, const float* view, const float* proj, int W, int H, int rect[4]);
/* row f3 (vr_parts.cu): k-d partition of the brick grid (0 = ok, 1 = more parts than the grid can be cut into) and the
 * parts front to back (0 = ok, 1 = singular view, 2 = malformed tree) */
int vr_host_kd_partition(int nx, int ny, int nz, int brick, int nparts, int* boxes_out, int* tree_out);
int vr_host_part_order(const int* tree, int nparts, int brick, const float* view, const float* proj, int* order_out);

#endif
