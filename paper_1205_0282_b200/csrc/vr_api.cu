/*
 * vr_api.cu -- the C ABI of libvr (include/vr.h): argument validation, device-memory
 * ownership, scratch sizing and kernel sequencing. No arithmetic of the method lives here;
 * every step of the path runs in the kernels of vr_bricks.cu, vr_setup.cu, vr_raycast.cu and
 * vr_composite.cu. There is no CPU fallback: without a CUDA device every call fails.
 */
#include <math.h>
#include <stdarg.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <new>

#include "vr_view.cuh"

static char g_err[512] = "no error";
static char* g_err_buf() { return g_err; }
/* for entry points that live in other files (vr_composite_static) */
void vr_global_error(const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
}

struct vr_volume {
    VrGrid grid;
    float* bricks;           /* nown * slot floats (nown = nbricks unless the handle is a part) */
    bool has_data, has_tf;
    float4* d_lut_base;      /* VR_MAX_LUT entries each */
    float4* d_lut_delta;
    VrLut lut;
    float tau;
    /* per-view scratch, written by the set-up kernel */
    VrViewState* d_vs;
    VrBrickView* d_bv;
    int* d_order;
    int* d_item_prefix;
    VrCompLayer* d_layers;
    void* d_sub;             /* sub-image scratch, sub_capacity_px * 16 bytes */
    long long sub_capacity_px;
    double2* d_rays;         /* the frame's ray table: VR_RAY_BYTES per pixel, ray_capacity_px pixels */
    long long ray_capacity_px;
    float* d_frame;          /* vr_render_host's device frame */
    long long frame_capacity_px;
    float* d_pipe[2];        /* vr_render_host_async: two device frames, ... */
    long long pipe_capacity_px;
    cudaStream_t copy_stream; /* ... a copy stream, and per frame slot: */
    cudaEvent_t ev_rendered[2], ev_copied[2];
    long long pipe_frames;
    float* d_stage;          /* staging for VR_HOST upload / download */
    long long stage_floats;
    int2* d_mm_enc;          /* row f1: per-brick range, order-preserving integer encoding */
    float2* d_mm;            /* nbricks + 1 entries: per brick, then the whole volume */
    int4* d_slot_ext;        /* nown entries: padded extent (x, y, z) of the brick in each slot */
    bool mm_valid;           /* d_mm describes the current contents of the store */
    float2* d_cell_mm;       /* R19: (min, max) per 8x8x8 macro-cell, nbricks * nc^3 (allocated on first use) */
    unsigned* d_cell_bits;   /* 1 = macro-cell transparent under the current LUT */
    int nc[3], cell_words;   /* macro-cells per axis of a slot; words of d_cell_bits per brick */
    bool cell_mm_valid, cell_bits_valid;
    bool mip_skip_known, mip_skip_useful; /* decided once per upload: does the cube have empty space (R19, MIP) */
    bool tex_alpha_known, tex_alpha_ok; /* decided per upload and transfer function: may ALPHA values come from the arrays at all (R20 vii) */
    float tf_slope;          /* largest difference between neighbouring table entries, in units of 1/n */
    float mean_cell_range;   /* mean (max - min) of the macro-cells, valid with tex_alpha_known */
    double* d_cell_stat;
    bool half_alpha_known, half_alpha_ok;  /* decided per upload and transfer function: may ALPHA values come from float16 texels (R22) */
    unsigned long long* d_cell_count;
    bool tf_smooth;          /* no neighbouring LUT entries further apart than 1.1/n per channel: no steeper than a full-range ramp (texture arm, R20) */
    bool tf_has_zero;        /* the LUT has a run of >= 3 zero-alpha entries: skipping can do something */
    bool culling;
    int sampler;             /* VR_SAMPLER_MANUAL or VR_SAMPLER_TEXTURE */
    VrTexStore* tex;         /* texture arm of the store (allocated by vr_set_sampler) */
    bool tex_valid;          /* the arrays hold the current contents of the store */
    VrVmm* vmm;              /* VR_LAYOUT_TILED_RELEASABLE: the store's physical memory, one chunk per slot */
    bool store_released;     /* vr_volume_release_store ran: only bricks with blanked voxels still have float32 cells */
    int traversal;           /* VR_SORT_LAST or VR_FUSED */
    int counting;            /* 0 off, 1 samples, 2 samples + touched-cells bitmap */
    bool timing;
    unsigned* d_bitmap;      /* one bit per brick-store cell (counting == 2) */
    long long bitmap_words;
    unsigned long long* d_counts2;
    cudaEvent_t ev[VR_EV_RING][4]; /* stage boundaries of the last VR_EV_RING timed frames */
    long long timed_frames;  /* frames rendered since timing was switched on */
    int last_W, last_H, last_mode;
    bool last_valid;       /* the last frame's sub-images are still in the scratch */
    bool last_stats_valid; /* the last frame's counters are still in the view state */
    int64_t launches;
    vr_alloc_fn alloc_fn;    /* the allocator in force when the handle was created (vr_set_allocator), or NULL = cudaMalloc */
    vr_free_fn free_fn;
    void* alloc_user;
    int* h_overflow;         /* mapped pinned flag the set-up kernel raises when a view needs more scratch than reserved */
    int* d_overflow;         /* its device address */
    char err[512];
};

/* process-wide allocator for handles created from now on (vr_set_allocator) */
static vr_alloc_fn g_alloc_fn = NULL;
static vr_free_fn g_free_fn = NULL;
static void* g_alloc_user = NULL;

extern "C" int vr_set_allocator(vr_alloc_fn alloc_fn, vr_free_fn free_fn, void* user) {
    if ((alloc_fn == NULL) != (free_fn == NULL)) {
        snprintf(g_err_buf(), 512, "vr_set_allocator: alloc and free must both be given, or both be NULL");
        return VR_ERR_INVALID_ARG;
    }
    g_alloc_fn = alloc_fn;
    g_free_fn = free_fn;
    g_alloc_user = user;
    return VR_OK;
}

/* device memory the handle owns: through the handle's allocator (torch's caching allocator in the Python binding) */
static cudaError_t v_alloc_bytes(const vr_volume* v, void** p, size_t bytes) {
    if (!v->alloc_fn) return cudaMalloc(p, bytes);
    *p = v->alloc_fn(bytes ? bytes : 1, v->alloc_user);
    return *p ? cudaSuccess : cudaErrorMemoryAllocation;
}
template <typename T>
static cudaError_t v_alloc(const vr_volume* v, T** p, size_t bytes) {
    return v_alloc_bytes(v, reinterpret_cast<void**>(p), bytes);
}
static void v_free(const vr_volume* v, void* p) {
    if (!p) return;
    if (v->free_fn) v->free_fn(p, v->alloc_user);
    else cudaFree(p);
}


static int fail(vr_volume* v, int status, const char* fmt, ...) {
    char* dst = v ? v->err : g_err;
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(dst, 512, fmt, ap);
    va_end(ap);
    return status;
}

#define VR_CUDA(v, call)                                                                                  \
    do {                                                                                                  \
        cudaError_t e_ = (call);                                                                          \
        if (e_ != cudaSuccess) {                                                                          \
            cudaGetLastError();                                                                           \
            return fail((v), e_ == cudaErrorMemoryAllocation ? VR_ERR_OUT_OF_MEMORY : VR_ERR_CUDA,        \
                        "%s failed: %s", #call, cudaGetErrorString(e_));                                  \
        }                                                                                                 \
    } while (0)

extern "C" const char* vr_last_error(const vr_volume* v) { return v ? v->err : g_err; }

extern "C" int vr_num_bricks(const vr_volume* v) { return v ? v->grid.nbricks : 0; }

extern "C" int64_t vr_launch_count(const vr_volume* v) { return v ? v->launches : 0; }

static void release(vr_volume* v) {
    vr_tex_destroy(v->tex);
    if (v->h_overflow) cudaFreeHost(v->h_overflow);
    if (v->vmm) vr_vmm_destroy(v->vmm);
    else v_free(v, v->bricks);
    v_free(v, v->d_lut_base);
    v_free(v, v->d_lut_delta);
    v_free(v, v->d_vs);
    v_free(v, v->d_bv);
    v_free(v, v->d_order);
    v_free(v, v->d_item_prefix);
    v_free(v, v->d_layers);
    v_free(v, v->d_sub);
    v_free(v, v->d_rays);
    v_free(v, v->d_frame);
    for (int i = 0; i < 2; ++i) {
        v_free(v, v->d_pipe[i]);
        if (v->ev_rendered[i]) cudaEventDestroy(v->ev_rendered[i]);
        if (v->ev_copied[i]) cudaEventDestroy(v->ev_copied[i]);
    }
    if (v->copy_stream) cudaStreamDestroy(v->copy_stream);
    v_free(v, v->d_stage);
    v_free(v, v->d_bitmap);
    v_free(v, v->d_mm_enc);
    v_free(v, v->d_mm);
    v_free(v, v->d_slot_ext);
    v_free(v, v->d_cell_mm);
    v_free(v, v->d_cell_bits);
    v_free(v, v->d_cell_count);
    v_free(v, v->d_cell_stat);
    v_free(v, v->d_counts2);
    for (int r = 0; r < VR_EV_RING; ++r)
        for (int i = 0; i < 4; ++i)
            if (v->ev[r][i]) cudaEventDestroy(v->ev[r][i]);
    cudaGetLastError();
    delete v;
}

extern "C" void vr_volume_destroy(vr_volume* v) {
    if (!v) return;
    cudaDeviceSynchronize();
    release(v);
}

/* Fill the layout part of the grid: per-axis offset functions and the slot size. */
static void set_layout(VrGrid& g, int layout, const int tl[3], const int ml[3]) {
    g.layout = layout;
    const int P = g.P;
    if (layout == VR_LAYOUT_LINEAR) {
        for (int a = 0; a < 3; ++a) {
            g.tl[a] = g.ml[a] = 0;
            g.nt[a] = P;
            VrAxisLayout& A = g.ax[a];
            memset(&A, 0, sizeof(A));
        }
        g.ax[0].lo_mask = 0x7fffffff; /* x: the index itself */
        g.ax[0].hi_in = 31;
        g.ax[1].hi_stride = (unsigned)P;
        g.ax[2].hi_stride = (unsigned)P * (unsigned)P;
        g.slot = (((long long)P * P * P + 31) / 32) * 32;
        return;
    }
    const int tbits = tl[0] + tl[1] + tl[2];          /* 5: 32 floats per micro-tile */
    const int mbits = ml[0] + ml[1] + ml[2];
    const unsigned block = 1u << (tbits + mbits);      /* floats per macro block */
    int lo_shift = 0, mid_shift = tbits;
    unsigned stride = block;
    for (int a = 0; a < 3; ++a) {
        g.tl[a] = tl[a];
        g.ml[a] = ml[a];
        const int span = 1 << (tl[a] + ml[a]);         /* cells per macro block along a */
        g.nt[a] = (P + span - 1) / span;
        VrAxisLayout& A = g.ax[a];
        A.lo_mask = (1 << tl[a]) - 1;
        A.lo_shift = lo_shift;
        A.mid_in = tl[a];
        A.mid_mask = (1 << ml[a]) - 1;
        A.mid_shift = mid_shift;
        A.hi_in = tl[a] + ml[a];
        A.hi_stride = stride;
        lo_shift += tl[a];
        mid_shift += ml[a];
        stride *= (unsigned)g.nt[a];
    }
    g.slot = (long long)block * g.nt[0] * g.nt[1] * g.nt[2];
}

extern "C" int vr_volume_create(int nx, int ny, int nz, int brick, int ghost, vr_volume** out) {
    return vr_volume_create_layout(nx, ny, nz, brick, ghost, VR_LAYOUT_DEFAULT, out);
}

static int create_volume(int nx, int ny, int nz, int brick, int ghost, int layout, const int* b0, const int* b1, vr_volume** out);

extern "C" int vr_volume_create_layout(int nx, int ny, int nz, int brick, int ghost, int layout, vr_volume** out) {
    return create_volume(nx, ny, nz, brick, ghost, layout, NULL, NULL, out);
}

extern "C" int vr_volume_create_part(int nx, int ny, int nz, int brick, int ghost, const int* b0, const int* b1, vr_volume** out) {
    if (!b0 || !b1) return fail(NULL, VR_ERR_INVALID_ARG, "vr_volume_create_part: NULL box");
    return create_volume(nx, ny, nz, brick, ghost, VR_LAYOUT_DEFAULT, b0, b1, out);
}

/* b0, b1: the box of bricks the handle holds (row f3), or NULL for the whole grid */
static int create_volume(int nx, int ny, int nz, int brick, int ghost, int layout, const int* b0, const int* b1, vr_volume** out) {
    if (!out) return fail(NULL, VR_ERR_INVALID_ARG, "vr_volume_create: out is NULL");
    *out = NULL;
    if (nx <= 0 || ny <= 0 || nz <= 0) return fail(NULL, VR_ERR_INVALID_ARG, "vr_volume_create: non-positive size %dx%dx%d", nx, ny, nz);
    if (brick < 2) return fail(NULL, VR_ERR_INVALID_ARG, "vr_volume_create: brick %d < 2", brick);
    if (ghost < 0 || ghost > 8) return fail(NULL, VR_ERR_INVALID_ARG, "vr_volume_create: ghost %d outside [0,8]", ghost);
    if (layout != VR_LAYOUT_DEFAULT && layout != VR_LAYOUT_LINEAR && layout != VR_LAYOUT_TILED && layout != VR_LAYOUT_TILED_RELEASABLE)
        return fail(NULL, VR_ERR_INVALID_ARG, "vr_volume_create_layout: unknown layout %d", layout);
    const bool releasable = layout == VR_LAYOUT_TILED_RELEASABLE;
    if (layout == VR_LAYOUT_DEFAULT || releasable) layout = VR_LAYOUT_TILED;
    if (releasable && g_alloc_fn) return fail(NULL, VR_ERR_STATE, "vr_volume_create_layout: a releasable store maps its own memory (vr_set_allocator is in force)");
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) {
        cudaGetLastError();
        return fail(NULL, VR_ERR_CUDA, "vr_volume_create: no CUDA device (libvr has no CPU path)");
    }
    vr_volume* v = new (std::nothrow) vr_volume();
    if (!v) return fail(NULL, VR_ERR_OUT_OF_MEMORY, "vr_volume_create: host allocation failed");
    memset(v, 0, sizeof(*v));
    snprintf(v->err, sizeof(v->err), "no error");
    VrGrid& g = v->grid;
    g.n[0] = nx; g.n[1] = ny; g.n[2] = nz;
    g.brick = brick; g.ghost = ghost;
    long long nb = 1;
    for (int a = 0; a < 3; ++a) {
        g.g[a] = (g.n[a] + brick - 1) / brick;
        nb *= g.g[a];
        if (g.g[a] > VR_MAX_AXIS_BRICKS) {
            delete v;
            return fail(NULL, VR_ERR_INVALID_ARG, "vr_volume_create: more than %d bricks along an axis", VR_MAX_AXIS_BRICKS);
        }
    }
    if (nb > 65535) {
        delete v;
        return fail(NULL, VR_ERR_INVALID_ARG, "vr_volume_create: %lld bricks > 65535", nb);
    }
    g.nbricks = (int)nb;
    g.part = 0;
    g.nown = g.nbricks;
    for (int a = 0; a < 3; ++a) g.pb0[a] = 0, g.pb1[a] = g.g[a];
    if (b0 && b1) {
        long long own = 1;
        for (int a = 0; a < 3; ++a) {
            if (b0[a] < 0 || b1[a] <= b0[a] || b1[a] > g.g[a]) {
                const int gx = g.g[0], gy = g.g[1], gz = g.g[2];
                delete v;
                return fail(NULL, VR_ERR_INVALID_ARG, "vr_volume_create_part: box [%d,%d) x [%d,%d) x [%d,%d) is empty or outside the %dx%dx%d brick grid",
                            b0[0], b1[0], b0[1], b1[1], b0[2], b1[2], gx, gy, gz);
            }
            g.pb0[a] = b0[a], g.pb1[a] = b1[a];
            own *= b1[a] - b0[a];
        }
        g.nown = (int)own;
        g.part = g.nown != g.nbricks;
    }
    /* a volume smaller than one brick needs no larger slot than itself */
    int core = brick;
    {
        int m = nx > ny ? nx : ny;
        m = m > nz ? m : nz;
        if (m < core) core = m;
    }
    g.P = core + 2 * ghost;
    g.brick_pow2 = (brick & (brick - 1)) == 0;
    {
        int tl[3] = {2, 2, 1}, ml[3] = {0, 0, 0};
        if (const char* e = getenv("VR_TILE")) { /* experiment knob: "lx,ly,lz,mx,my,mz" (log2) */
            const int got = sscanf(e, "%d,%d,%d,%d,%d,%d", &tl[0], &tl[1], &tl[2], &ml[0], &ml[1], &ml[2]);
            bool ok = got == 6 && tl[0] + tl[1] + tl[2] == 5; /* a micro-tile is 32 floats = one 128-byte line */
            for (int a = 0; a < 3; ++a) ok = ok && tl[a] >= 0 && tl[a] <= 5 && ml[a] >= 0 && ml[a] <= 4;
            if (!ok) {
                delete v;
                return fail(NULL, VR_ERR_INVALID_ARG, "vr_volume_create: VR_TILE=\"%s\" is not six log2 sizes with lx+ly+lz = 5, m* in [0,4]", e);
            }
        }
        if (const char* e = getenv("VR_LAYOUT")) {
            if (strcmp(e, "1") != 0 && strcmp(e, "2") != 0) {
                delete v;
                return fail(NULL, VR_ERR_INVALID_ARG, "vr_volume_create: VR_LAYOUT=\"%s\" is neither 1 (linear) nor 2 (tiled)", e);
            }
            layout = e[0] == '1' ? VR_LAYOUT_LINEAR : VR_LAYOUT_TILED;
        }
        set_layout(g, layout, tl, ml);
    }
    if (g.slot >= (1ll << 31)) {
        delete v;
        return fail(NULL, VR_ERR_INVALID_ARG, "vr_volume_create: a padded brick of %d^3 cells exceeds 2^31 floats", g.P);
    }
    v->tau = 0.99f;
    v->culling = true;
    v->alloc_fn = g_alloc_fn;
    v->free_fn = g_free_fn;
    v->alloc_user = g_alloc_user;

    cudaError_t e;
    if (releasable) {
        e = vr_vmm_create((size_t)g.slot * sizeof(float), g.nown, &v->vmm, &v->bricks);
        if (e == cudaErrorNotSupported) {
            cudaGetLastError();
            delete v;
            return fail(NULL, VR_ERR_CUDA, "vr_volume_create_layout: no CUDA virtual memory management on this device or driver");
        }
    } else {
        e = v_alloc(v, &v->bricks, (size_t)g.slot * (size_t)g.nown * sizeof(float));
    }
    if (e == cudaSuccess) e = cudaMemset(v->bricks, 0, (size_t)g.slot * (size_t)g.nown * sizeof(float));
    if (e == cudaSuccess) e = v_alloc(v, &v->d_lut_base, VR_MAX_LUT * sizeof(float4));
    if (e == cudaSuccess) e = v_alloc(v, &v->d_lut_delta, VR_MAX_LUT * sizeof(float4));
    if (e == cudaSuccess) e = v_alloc(v, &v->d_vs, sizeof(VrViewState));
    if (e == cudaSuccess) e = cudaMemset(v->d_vs, 0, sizeof(VrViewState));
    if (e == cudaSuccess) e = v_alloc(v, &v->d_bv, sizeof(VrBrickView) * g.nbricks);
    if (e == cudaSuccess) e = v_alloc(v, &v->d_order, sizeof(int) * g.nbricks);
    if (e == cudaSuccess) e = v_alloc(v, &v->d_item_prefix, sizeof(int) * (g.nbricks + 1));
    if (e == cudaSuccess) e = v_alloc(v, &v->d_layers, sizeof(VrCompLayer) * g.nbricks);
    if (e == cudaSuccess) e = v_alloc(v, &v->d_mm_enc, sizeof(int2) * g.nbricks);
    if (e == cudaSuccess) e = v_alloc(v, &v->d_mm, sizeof(float2) * (g.nbricks + 1));
    for (int r = 0; r < VR_EV_RING && e == cudaSuccess; ++r)
        for (int i = 0; i < 4 && e == cudaSuccess; ++i) e = cudaEventCreate(&v->ev[r][i]);
    if (e == cudaSuccess) e = v_alloc(v, &v->d_slot_ext, sizeof(int4) * g.nown);
    if (e == cudaSuccess) {
        int4* ext = new (std::nothrow) int4[g.nown];
        if (!ext) e = cudaErrorMemoryAllocation;
        for (int b = 0; ext && b < g.nbricks; ++b) {
            const int s = vr_slot_index(g, b);
            if (s < 0) continue;
            int bc[3], lo[3], hi[3];
            vr_brick_coords(g, b, bc);
            vr_brick_core(g, bc, lo, hi);
            ext[s] = make_int4(hi[0] - lo[0] + 2 * ghost, hi[1] - lo[1] + 2 * ghost, hi[2] - lo[2] + 2 * ghost, b);
        }
        if (ext) e = cudaMemcpy(v->d_slot_ext, ext, sizeof(int4) * g.nown, cudaMemcpyHostToDevice);
        delete[] ext;
    }
    if (e == cudaSuccess) e = cudaHostAlloc(&v->h_overflow, sizeof(int), cudaHostAllocMapped);
    if (e == cudaSuccess) {
        *v->h_overflow = 0;
        e = cudaHostGetDevicePointer(&v->d_overflow, v->h_overflow, 0);
    }
    if (e != cudaSuccess) {
        cudaGetLastError();
        const int st = (e == cudaErrorMemoryAllocation) ? VR_ERR_OUT_OF_MEMORY : VR_ERR_CUDA;
        fail(NULL, st, "vr_volume_create: %s (brick store needs %.2f GB)", cudaGetErrorString(e),
             (double)g.slot * g.nown * 4.0 / 1e9);
        release(v);
        return st;
    }
    *out = v;
    return VR_OK;
}

static int check_box(vr_volume* v, const char* who, const void* p, int memspace, int x0, int y0, int z0, int sx, int sy, int sz) {
    if (!v) return fail(NULL, VR_ERR_INVALID_ARG, "%s: NULL handle", who);
    if (!p) return fail(v, VR_ERR_INVALID_ARG, "%s: NULL data pointer", who);
    if (memspace != VR_HOST && memspace != VR_DEVICE) return fail(v, VR_ERR_INVALID_ARG, "%s: bad memspace %d", who, memspace);
    if (sx <= 0 || sy <= 0 || sz <= 0) return fail(v, VR_ERR_INVALID_ARG, "%s: empty box %dx%dx%d", who, sx, sy, sz);
    const VrGrid& g = v->grid;
    if (x0 < 0 || y0 < 0 || z0 < 0 || (long long)x0 + sx > g.n[0] || (long long)y0 + sy > g.n[1] || (long long)z0 + sz > g.n[2])
        return fail(v, VR_ERR_INVALID_ARG, "%s: box (%d,%d,%d)+(%d,%d,%d) outside the %dx%dx%d volume", who, x0, y0, z0, sx, sy,
                    sz, g.n[0], g.n[1], g.n[2]);
    return VR_OK;
}

/* planes of an [sy][sx] box per staging chunk: at most 256 MiB, at least one plane */
static int ensure_stage(vr_volume* v, int sx, int sy, int sz, int* planes) {
    const long long plane = (long long)sx * sy;
    long long n = (64ll << 20) / plane;
    if (n < 1) n = 1;
    if (n > sz) n = sz;
    if (v->stage_floats < n * plane) {
        if (v->d_stage) {
            cudaDeviceSynchronize();
            v_free(v, v->d_stage);
            v->d_stage = NULL;
            v->stage_floats = 0;
        }
        VR_CUDA(v, v_alloc(v, &v->d_stage, (size_t)(n * plane) * sizeof(float)));
        v->stage_floats = n * plane;
    }
    *planes = (int)n;
    return VR_OK;
}

extern "C" int vr_volume_upload(vr_volume* v, const float* src, int memspace, int x0, int y0, int z0, int sx, int sy, int sz,
                                void* stream) {
    int rc = check_box(v, "vr_volume_upload", src, memspace, x0, y0, z0, sx, sy, sz);
    if (rc) return rc;
    if (v->store_released) return fail(v, VR_ERR_STATE, "vr_volume_upload: the float32 store was released (vr_volume_release_store)");
    cudaStream_t st = (cudaStream_t)stream;
    if (memspace == VR_DEVICE) {
        VR_CUDA(v, vr_launch_upload(v->grid, v->bricks, src, x0, y0, z0, sx, sy, sz, st));
        v->launches++;
    } else {
        int planes = 0;
        rc = ensure_stage(v, sx, sy, sz, &planes);
        if (rc) return rc;
        const long long plane = (long long)sx * sy;
        for (int k = 0; k < sz; k += planes) {
            const int nk = (sz - k < planes) ? sz - k : planes;
            VR_CUDA(v, cudaMemcpyAsync(v->d_stage, src + (long long)k * plane, (size_t)(nk * plane) * sizeof(float),
                                       cudaMemcpyHostToDevice, st));
            VR_CUDA(v, vr_launch_upload(v->grid, v->bricks, v->d_stage, x0, y0, z0 + k, sx, sy, nk, st));
            v->launches++;
            VR_CUDA(v, cudaStreamSynchronize(st)); /* the staging buffer is reused */
        }
    }
    v->has_data = true;
    v->tex_valid = false;
    v->mm_valid = false;
    v->cell_mm_valid = v->cell_bits_valid = false;
    v->mip_skip_known = false;
    v->half_alpha_known = false;
    v->tex_alpha_known = false;
    return VR_OK;
}

extern "C" int vr_volume_download(vr_volume* v, float* dst, int memspace, int x0, int y0, int z0, int sx, int sy, int sz,
                                  void* stream) {
    int rc = check_box(v, "vr_volume_download", dst, memspace, x0, y0, z0, sx, sy, sz);
    if (rc) return rc;
    if (v->store_released) return fail(v, VR_ERR_STATE, "vr_volume_download: the float32 store was released (vr_volume_release_store)");
    if (v->grid.part) { /* a part can return voxels of its own bricks only */
        const VrGrid& g = v->grid;
        const int lo[3] = {x0, y0, z0}, hi[3] = {x0 + sx, y0 + sy, z0 + sz};
        for (int a = 0; a < 3; ++a) {
            const long long plo = (long long)g.pb0[a] * g.brick, phi = (long long)g.pb1[a] * g.brick;
            if (lo[a] < plo || hi[a] > (phi < g.n[a] ? phi : g.n[a]))
                return fail(v, VR_ERR_INVALID_ARG, "vr_volume_download: the box leaves the bricks this part holds");
        }
    }
    cudaStream_t st = (cudaStream_t)stream;
    if (memspace == VR_DEVICE) {
        VR_CUDA(v, vr_launch_download(v->grid, v->bricks, dst, x0, y0, z0, sx, sy, sz, st));
        v->launches++;
        return VR_OK;
    }
    int planes = 0;
    rc = ensure_stage(v, sx, sy, sz, &planes);
    if (rc) return rc;
    const long long plane = (long long)sx * sy;
    for (int k = 0; k < sz; k += planes) {
        const int nk = (sz - k < planes) ? sz - k : planes;
        VR_CUDA(v, vr_launch_download(v->grid, v->bricks, v->d_stage, x0, y0, z0 + k, sx, sy, nk, st));
        v->launches++;
        VR_CUDA(v, cudaMemcpyAsync(dst + (long long)k * plane, v->d_stage, (size_t)(nk * plane) * sizeof(float),
                                   cudaMemcpyDeviceToHost, st));
        VR_CUDA(v, cudaStreamSynchronize(st));
    }
    return VR_OK;
}

extern "C" int vr_debug_set_upload_path(int path) {
    if (path != 0 && path != 1) return fail(NULL, VR_ERR_INVALID_ARG, "vr_debug_set_upload_path: 0 (cp.async) or 1 (TMA)");
    vr_set_upload_path(path);
    return VR_OK;
}

extern "C" int vr_debug_brick_data(vr_volume* v, int b, float* dst, int* dims) {
    if (!v) return fail(NULL, VR_ERR_INVALID_ARG, "vr_debug_brick_data: NULL handle");
    const VrGrid& g = v->grid;
    if (b < 0 || b >= g.nbricks || !dims) return fail(v, VR_ERR_INVALID_ARG, "vr_debug_brick_data: bad brick %d or NULL dims", b);
    if (vr_slot_index(g, b) < 0) return fail(v, VR_ERR_INVALID_ARG, "vr_debug_brick_data: this part does not hold brick %d", b);
    if (v->store_released) return fail(v, VR_ERR_STATE, "vr_debug_brick_data: the float32 store was released (vr_volume_release_store)");
    const int bx = b % g.g[0], by = (b / g.g[0]) % g.g[1], bz = b / (g.g[0] * g.g[1]);
    const int bc[3] = {bx, by, bz};
    int d[3];
    for (int a = 0; a < 3; ++a) {
        const int lo = bc[a] * g.brick;
        int hi = lo + g.brick;
        if (hi > g.n[a]) hi = g.n[a];
        d[a] = hi - lo + 2 * g.ghost;
        dims[a] = d[a];
    }
    if (!dst) return VR_OK;
    VR_CUDA(v, cudaDeviceSynchronize());
    float* d_tmp = NULL;
    const size_t bytes = (size_t)d[0] * d[1] * d[2] * sizeof(float);
    VR_CUDA(v, cudaMalloc(&d_tmp, bytes));
    cudaError_t e = vr_launch_brick_copy(g, v->bricks, b, d, d_tmp, 0);
    v->launches++;
    if (e == cudaSuccess) e = cudaMemcpy(dst, d_tmp, bytes, cudaMemcpyDeviceToHost);
    cudaFree(d_tmp);
    VR_CUDA(v, e);
    return VR_OK;
}

/* ------------------------------------------------------------------------------------------ */
extern "C" int vr_set_transfer_function(vr_volume* v, const float* rgba, int n, float vmin, float vmax) {
    if (!v) return fail(NULL, VR_ERR_INVALID_ARG, "vr_set_transfer_function: NULL handle");
    if (!rgba) return fail(v, VR_ERR_INVALID_ARG, "vr_set_transfer_function: NULL table");
    if (n < 2 || n > VR_MAX_LUT) return fail(v, VR_ERR_INVALID_ARG, "vr_set_transfer_function: n = %d outside [2,%d]", n, VR_MAX_LUT);
    if (!(vmax > vmin) || !isfinite(vmin) || !isfinite(vmax))
        return fail(v, VR_ERR_INVALID_ARG, "vr_set_transfer_function: need finite vmin < vmax");
    for (int i = 0; i < 4 * n; ++i)
        if (!isfinite(rgba[i])) return fail(v, VR_ERR_INVALID_ARG, "vr_set_transfer_function: entry %d is not finite", i / 4);
    for (int i = 0; i < n; ++i) /* R7: the table's alpha is an opacity; log2(1 - a) of anything else is NaN */
        if (!(rgba[4 * i + 3] >= 0.0f && rgba[4 * i + 3] <= 1.0f))
            return fail(v, VR_ERR_INVALID_ARG, "vr_set_transfer_function: alpha %g of entry %d outside [0,1]", rgba[4 * i + 3], i);
    /* the table is stored as (entry, difference to the next entry) pairs; the differences are
     * plain float32 subtractions of the caller's entries */
    float4 base[VR_MAX_LUT], delta[VR_MAX_LUT]; /* 32 KB of stack: no state shared between handles or threads */
    for (int i = 0; i < n; ++i) {
        base[i] = make_float4(rgba[4 * i], rgba[4 * i + 1], rgba[4 * i + 2], rgba[4 * i + 3]);
        if (i + 1 < n)
            delta[i] = make_float4(rgba[4 * i + 4] - rgba[4 * i], rgba[4 * i + 5] - rgba[4 * i + 1],
                                   rgba[4 * i + 6] - rgba[4 * i + 2], rgba[4 * i + 7] - rgba[4 * i + 3]);
        else
            delta[i] = make_float4(0.f, 0.f, 0.f, 0.f);
    }
    VR_CUDA(v, cudaDeviceSynchronize());
    VR_CUDA(v, cudaMemcpy(v->d_lut_base, base, sizeof(float4) * n, cudaMemcpyHostToDevice));
    VR_CUDA(v, cudaMemcpy(v->d_lut_delta, delta, sizeof(float4) * n, cudaMemcpyHostToDevice));
    v->lut.base = v->d_lut_base;
    v->lut.delta = v->d_lut_delta;
    v->lut.n = n;
    v->lut.vmin = vmin;
    v->lut.vmax = vmax;
    v->lut.inv_range = (float)(1.0 / ((double)vmax - (double)vmin));
    v->lut.nm2 = n - 2;
    v->lut.scale = (float)(n - 1);
    /* R16 needs every entry of [I(min)-1, I(max)+2] transparent: at least three consecutive zero-alpha entries
     * (a lone zero at entry 0, as in a linear ramp, can never make anything transparent) */
    v->tf_has_zero = false;
    for (int i = 0, run = 0; i < n; ++i) {
        run = rgba[4 * i + 3] == 0.0f ? run + 1 : 0;
        if (run >= 3) v->tf_has_zero = true;
    }
    /* texture arm: the filter's 8-bit weights put a value error of up to ~3 * 2^-9 of the local voxel differences on a
     * sample (about one table entry on noise of unit sigma over a 13-sigma, 256-entry table); 2e-3 per channel survives that
     * only if neighbouring entries are close. Tables with steps (thresholds, toes) keep the hand-rolled sampler. */
    v->tf_smooth = true;
    v->tf_slope = 0.0f;
    v->half_alpha_known = false;
    v->tex_alpha_known = false;
    for (int i = 0; i + 1 < n; ++i)
        for (int c = 0; c < 4; ++c) {
            v->tf_slope = fmaxf(v->tf_slope, fabsf(rgba[4 * i + 4 + c] - rgba[4 * i + c]) * (float)n);
            if (fabsf(rgba[4 * i + 4 + c] - rgba[4 * i + c]) > 1.1f / (float)n) v->tf_smooth = false; /* R20 (ii): no steeper than a full-range ramp */
        }
    v->cell_bits_valid = false;
    v->has_tf = true;
    return VR_OK;
}

extern "C" int vr_set_early_termination(vr_volume* v, float tau) {
    if (!v) return fail(NULL, VR_ERR_INVALID_ARG, "vr_set_early_termination: NULL handle");
    if (!(tau > 0.0f)) return fail(v, VR_ERR_INVALID_ARG, "vr_set_early_termination: tau must be > 0");
    v->tau = tau;
    return VR_OK;
}

extern "C" int vr_set_counting(vr_volume* v, int enable) {
    if (!v) return fail(NULL, VR_ERR_INVALID_ARG, "vr_set_counting: NULL handle");
    if (enable < 0 || enable > 2) return fail(v, VR_ERR_INVALID_ARG, "vr_set_counting: mode %d outside [0,2]", enable);
    if (enable == 2 && !v->d_bitmap) {
        const long long words = (v->grid.slot * v->grid.nown + 31) / 32;
        VR_CUDA(v, v_alloc(v, &v->d_bitmap, (size_t)words * sizeof(unsigned)));
        VR_CUDA(v, v_alloc(v, &v->d_counts2, 3 * sizeof(unsigned long long)));
        v->bitmap_words = words;
    }
    v->counting = enable;
    return VR_OK;
}

extern "C" int vr_set_timing(vr_volume* v, int enable) {
    if (!v) return fail(NULL, VR_ERR_INVALID_ARG, "vr_set_timing: NULL handle");
    v->timing = enable != 0;
    v->timed_frames = 0;
    return VR_OK;
}

/* ------------------------------------------------------------------------------------------ */
static int check_view(vr_volume* v, const char* who, const float* view, const float* proj, int W, int H, long long* sub_px,
                      long long* items) {
    if (!v) return fail(NULL, VR_ERR_INVALID_ARG, "%s: NULL handle", who);
    if (!view || !proj) return fail(v, VR_ERR_INVALID_ARG, "%s: NULL matrix", who);
    if (W <= 0 || H <= 0 || W > 32768 || H > 32768) return fail(v, VR_ERR_INVALID_ARG, "%s: bad frame size %dx%d", who, W, H);
    for (int i = 0; i < 16; ++i)
        if (!isfinite(view[i]) || !isfinite(proj[i])) return fail(v, VR_ERR_INVALID_ARG, "%s: matrix entry is not finite", who);
    if (vr_host_view_check(v->grid, view, proj, W, H, sub_px, items))
        return fail(v, VR_ERR_INVALID_ARG, "%s: proj*view is singular", who);
    if (*items > 2000000000ll) return fail(v, VR_ERR_INVALID_ARG, "%s: view needs %lld work items (> 2e9)", who, *items);
    return VR_OK;
}

/* A view that needed more sub-image scratch than was reserved (host and device rectangle arithmetic disagreed by more
 * than the slack, or vr_reserve_views was given other views) renders a blank frame and raises a flag in mapped host
 * memory: the next call on the handle that looks reports it. */
static int check_overflow(vr_volume* v, const char* who) {
    if (v->h_overflow && *(volatile int*)v->h_overflow) {
        *v->h_overflow = 0;
        return fail(v, VR_ERR_STATE, "%s: an earlier frame needed more sub-image scratch than was reserved and came out blank", who);
    }
    return VR_OK;
}

static int ensure_sub(vr_volume* v, long long need_px) {
    if (need_px <= v->sub_capacity_px) return VR_OK;
    if (v->d_sub) {
        VR_CUDA(v, cudaDeviceSynchronize());
        v_free(v, v->d_sub);
        v->d_sub = NULL;
        v->sub_capacity_px = 0;
    }
    const long long cap = need_px + need_px / 4 + 4096; /* headroom: neighbouring views fit too */
    VR_CUDA(v, v_alloc(v, &v->d_sub, (size_t)cap * 16));
    v->sub_capacity_px = cap;
    return VR_OK;
}

/* The ray table of a W x H frame (vr_rays.cu). */
static int ensure_rays(vr_volume* v, long long px) {
    if (px <= v->ray_capacity_px) return VR_OK;
    if (v->d_rays) {
        VR_CUDA(v, cudaDeviceSynchronize());
        v_free(v, v->d_rays);
        v->d_rays = NULL;
        v->ray_capacity_px = 0;
    }
    VR_CUDA(v, v_alloc(v, &v->d_rays, (size_t)px * VR_RAY_BYTES + 16));
    v->ray_capacity_px = px;
    return VR_OK;
}

/* vr_render_host_async's two device frames, copy stream and events, for frames of px pixels */
static int ensure_pipe(vr_volume* v, long long px) {
    if (!v->copy_stream) {
        VR_CUDA(v, cudaStreamCreateWithFlags(&v->copy_stream, cudaStreamNonBlocking));
        for (int i = 0; i < 2; ++i) {
            VR_CUDA(v, cudaEventCreateWithFlags(&v->ev_rendered[i], cudaEventDisableTiming));
            VR_CUDA(v, cudaEventCreateWithFlags(&v->ev_copied[i], cudaEventDisableTiming));
        }
    }
    if (px > v->pipe_capacity_px) {
        VR_CUDA(v, cudaDeviceSynchronize());
        for (int i = 0; i < 2; ++i) {
            v_free(v, v->d_pipe[i]);
            v->d_pipe[i] = NULL;
        }
        v->pipe_capacity_px = 0;
        for (int i = 0; i < 2; ++i) VR_CUDA(v, v_alloc(v, &v->d_pipe[i], (size_t)px * 16));
        v->pipe_capacity_px = px;
    }
    return VR_OK;
}

/* Row f1: bring the range table up to date with the store (three launches, after an upload only). */
static bool cells_supported(const vr_volume* v);
static int alloc_cells(vr_volume* v);

static int ensure_minmax(vr_volume* v, cudaStream_t st) {
    if (v->mm_valid) return VR_OK;
    if (cells_supported(v)) { /* the macro-cell table (R19) comes out of the same read of the store */
        const int rc = alloc_cells(v);
        if (rc) return rc;
        VR_CUDA(v, vr_launch_ranges(v->grid, v->bricks, v->d_mm_enc, v->d_mm, v->d_cell_mm, v->nc, v->d_slot_ext, st));
        v->launches += 4;
        v->cell_mm_valid = true;
        v->cell_bits_valid = false;
    } else {
        VR_CUDA(v, vr_launch_minmax(v->grid, v->bricks, v->d_mm_enc, v->d_mm, st));
        v->launches += 3;
    }
    v->mm_valid = true;
    return VR_OK;
}

/* R19: macro-cell ranges (after an upload) and transparency bits (after an upload or a new transfer
 * function). Only for the 4x4x2 layout with ghost cells; memory is taken on first use. */
static bool cells_supported(const vr_volume* v) {
    const VrGrid& g = v->grid;
    return g.layout == VR_LAYOUT_TILED && g.tl[0] == 2 && g.tl[1] == 2 && g.tl[2] == 1 && g.ml[0] == 0 && g.ml[1] == 0 &&
           g.ml[2] == 0 && g.ghost >= 1;
}

/* memory of the macro-cell tables (taken on first use, or ahead of it by vr_reserve_views) */
static int alloc_cells(vr_volume* v) {
    const VrGrid& g = v->grid;
    if (!v->d_cell_mm) {
        for (int a = 0; a < 3; ++a) v->nc[a] = (g.nt[a] * (1 << g.tl[a]) + 7) / 8;
        const long long ncell = (long long)v->nc[0] * v->nc[1] * v->nc[2];
        v->cell_words = (int)((ncell + 31) / 32);
        VR_CUDA(v, v_alloc(v, &v->d_cell_mm, sizeof(float2) * (size_t)ncell * g.nown));
        VR_CUDA(v, v_alloc(v, &v->d_cell_bits, sizeof(unsigned) * (size_t)v->cell_words * g.nown));
    }
    if (!v->d_cell_count) VR_CUDA(v, v_alloc(v, &v->d_cell_count, sizeof(unsigned long long)));
    return VR_OK;
}

static int ensure_cells(vr_volume* v, bool want_bits, cudaStream_t st) {
    const VrGrid& g = v->grid;
    {
        const int rc = alloc_cells(v);
        if (rc) return rc;
    }
    if (!v->cell_mm_valid) {
        VR_CUDA(v, vr_launch_cell_minmax(g, v->bricks, v->d_cell_mm, v->nc, st));
        v->launches++;
        v->cell_mm_valid = true;
        v->cell_bits_valid = false;
    }
    if (want_bits && !v->cell_bits_valid) {
        VR_CUDA(v, vr_launch_cell_flags(v->d_cell_mm, v->d_cell_bits, g.nown, v->nc, v->cell_words, v->lut, st));
        v->launches++;
        v->cell_bits_valid = true;
    }
    return VR_OK;
}

/* MIP (R19): stepping over macro-cells that cannot raise a ray's maximum pays only if the cube has empty
 * space - macro-cells that hold nothing but the global minimum (the zero background of a density cube).
 * Decided once per upload (one pass over the cell table and one 8-byte read-back): at least an eighth. */
static int decide_mip_skip(vr_volume* v, cudaStream_t st) {
    if (v->mip_skip_known) return VR_OK;
    int rc = ensure_minmax(v, st);
    if (!rc) rc = ensure_cells(v, false, st);
    if (rc) return rc;
    const long long ncells = (long long)v->nc[0] * v->nc[1] * v->nc[2] * v->grid.nown;
    unsigned long long empty = 0;
    VR_CUDA(v, cudaMemsetAsync(v->d_cell_count, 0, sizeof(unsigned long long), st));
    VR_CUDA(v, vr_launch_cell_count_empty(v->d_cell_mm, ncells, v->d_mm + v->grid.nbricks, v->d_cell_count, st));
    v->launches++;
    VR_CUDA(v, cudaMemcpyAsync(&empty, v->d_cell_count, sizeof(empty), cudaMemcpyDeviceToHost, st));
    VR_CUDA(v, cudaStreamSynchronize(st));
    v->mip_skip_useful = empty * 8ull >= (unsigned long long)ncells;
    v->mip_skip_known = true;
    return VR_OK;
}

/* R20 (vii): the filter's error is proportional to the voxel-to-voxel differences against the table's range. The mean range of
 * the 8x8x8 macro-cells stands for those differences; measured on the benchmark cubes (ratio R = mean cell range / table range =
 * 0.46-0.48, ramp table: slope 1) the largest pixel error of a frame is 1.4e-3 to 1.65e-3, i.e. up to 3.5e-3 x R x slope. ALPHA values
 * come from the arrays only while that estimate stays below 1.9e-3; decided once per upload / table. */
static int decide_tex_alpha(vr_volume* v, cudaStream_t st) {
    if (v->tex_alpha_known) return VR_OK;
    v->tex_alpha_ok = false;
    v->mean_cell_range = 0.0f;
    if (cells_supported(v)) {
        int rc = ensure_minmax(v, st);
        if (rc) return rc;
        if (!v->d_cell_stat) VR_CUDA(v, v_alloc(v, &v->d_cell_stat, 2 * sizeof(double)));
        const long long ncells = (long long)v->nc[0] * v->nc[1] * v->nc[2] * v->grid.nown;
        double stat[2] = {0.0, 0.0};
        VR_CUDA(v, cudaMemsetAsync(v->d_cell_stat, 0, sizeof(stat), st));
        VR_CUDA(v, vr_launch_cell_range_sum(v->d_cell_mm, ncells, v->d_cell_stat, st));
        v->launches++;
        VR_CUDA(v, cudaMemcpyAsync(stat, v->d_cell_stat, sizeof(stat), cudaMemcpyDeviceToHost, st));
        VR_CUDA(v, cudaStreamSynchronize(st));
        if (stat[1] > 0.0) {
            v->mean_cell_range = (float)(stat[0] / stat[1]);
            const float R = v->mean_cell_range / (v->lut.vmax - v->lut.vmin);
            v->tex_alpha_ok = 3.5e-3f * R * v->tf_slope <= 1.9e-3f;
        }
    }
    v->tex_alpha_known = true;
    return VR_OK;
}

/* R22: float16 texels move a value by up to 2^-10 of its magnitude (rounding + the unit's float16 filter). ALPHA frames
 * take their values from such arrays only while that stays below 1.5e-3 of the transfer function's range for the
 * largest magnitude in the volume (about a third of an entry of a 256-entry table); decided once per upload / table. */
static int decide_half_alpha(vr_volume* v, cudaStream_t st) {
    if (v->half_alpha_known) return VR_OK;
    const int rc = ensure_minmax(v, st);
    if (rc) return rc;
    float2 mm;
    VR_CUDA(v, cudaMemcpyAsync(&mm, v->d_mm + v->grid.nbricks, sizeof(mm), cudaMemcpyDeviceToHost, st));
    VR_CUDA(v, cudaStreamSynchronize(st));
    const float mag = fmaxf(fabsf(mm.x), fabsf(mm.y));
    v->half_alpha_ok = mag * (1.0f / 1024.0f) <= 1.5e-3f * (v->lut.vmax - v->lut.vmin); /* false for NaN / inf too */
    v->half_alpha_known = true;
    return VR_OK;
}

static int run_setup(vr_volume* v, const float* view, const float* proj, int W, int H, int mode, bool use_range,
                     cudaStream_t st) {
    VrMatrices m;
    memcpy(m.view, view, sizeof(m.view));
    memcpy(m.proj, proj, sizeof(m.proj));
    if (use_range) {
        const int rc = ensure_minmax(v, st);
        if (rc) return rc;
    }
    VR_CUDA(v, vr_launch_setup(v->grid, m, W, H, mode, v->sub_capacity_px, v->d_sub, v->d_vs, v->d_bv, v->d_order,
                               v->d_item_prefix, v->d_layers, use_range ? v->d_mm : NULL, v->lut, v->d_overflow, st));
    v->launches++;
    return VR_OK;
}

extern "C" int vr_reserve_views(vr_volume* v, const float* views, const float* projs, int nviews, int width, int height) {
    if (!v) return fail(NULL, VR_ERR_INVALID_ARG, "vr_reserve_views: NULL handle");
    if (nviews < 0 || (nviews > 0 && (!views || !projs))) return fail(v, VR_ERR_INVALID_ARG, "vr_reserve_views: NULL matrices");
    if (width <= 0 || height <= 0 || width > 32768 || height > 32768)
        return fail(v, VR_ERR_INVALID_ARG, "vr_reserve_views: bad frame size %dx%d", width, height);
    long long need = 0;
    for (int q = 0; q < nviews; ++q) {
        long long sub_px = 0, items = 0;
        const int rc = check_view(v, "vr_reserve_views", views + 16 * q, projs + 16 * q, width, height, &sub_px, &items);
        if (rc) return rc;
        if (sub_px > need) need = sub_px;
    }
    const long long px = (long long)width * height;
    int rc = ensure_sub(v, need > 0 ? need : px);
    if (!rc) rc = ensure_rays(v, px);
    if (!rc && cells_supported(v)) rc = alloc_cells(v); /* R19's tables: filled by the first frame that uses them */
    if (rc) return rc;
    /* the host entries' device frames (vr_render_host: one; vr_render_host_async: two, a stream and four events) */
    if (px > v->frame_capacity_px) {
        if (v->d_frame) {
            VR_CUDA(v, cudaDeviceSynchronize());
            v_free(v, v->d_frame);
            v->d_frame = NULL;
            v->frame_capacity_px = 0;
        }
        VR_CUDA(v, v_alloc(v, &v->d_frame, (size_t)px * 16));
        v->frame_capacity_px = px;
    }
    return ensure_pipe(v, px);
}

extern "C" int vr_volume_minmax(vr_volume* v, float* vmin_out, float* vmax_out, void* stream) {
    if (!v) return fail(NULL, VR_ERR_INVALID_ARG, "vr_volume_minmax: NULL handle");
    if (!vmin_out || !vmax_out) return fail(v, VR_ERR_INVALID_ARG, "vr_volume_minmax: NULL output");
    if (!v->has_data) return fail(v, VR_ERR_STATE, "vr_volume_minmax: nothing uploaded");
    cudaStream_t st = (cudaStream_t)stream;
    const int rc = ensure_minmax(v, st);
    if (rc) return rc;
    float2 mm;
    VR_CUDA(v, cudaMemcpyAsync(&mm, v->d_mm + v->grid.nbricks, sizeof(mm), cudaMemcpyDeviceToHost, st));
    VR_CUDA(v, cudaStreamSynchronize(st));
    *vmin_out = mm.x;
    *vmax_out = mm.y;
    return VR_OK;
}

extern "C" int vr_set_traversal(vr_volume* v, int traversal) {
    if (!v) return fail(NULL, VR_ERR_INVALID_ARG, "vr_set_traversal: NULL handle");
    if (traversal != VR_SORT_LAST && traversal != VR_FUSED)
        return fail(v, VR_ERR_INVALID_ARG, "vr_set_traversal: unknown traversal %d", traversal);
    v->traversal = traversal;
    return VR_OK;
}

extern "C" int vr_set_sampler(vr_volume* v, int sampler) {
    if (!v) return fail(NULL, VR_ERR_INVALID_ARG, "vr_set_sampler: NULL handle");
    if (sampler != VR_SAMPLER_MANUAL && sampler != VR_SAMPLER_TEXTURE && sampler != VR_SAMPLER_TEXTURE_HALF && sampler != VR_SAMPLER_TEXTURE_BYTE)
        return fail(v, VR_ERR_INVALID_ARG, "vr_set_sampler: unknown sampler %d", sampler);
    if (v->store_released && sampler != v->sampler)
        return fail(v, VR_ERR_STATE, "vr_set_sampler: the float32 store was released, only the arrays it was turned into are left");
    const int texel = sampler == VR_SAMPLER_TEXTURE_HALF ? VR_TEXEL_HALF : sampler == VR_SAMPLER_TEXTURE_BYTE ? VR_TEXEL_BYTE : VR_TEXEL_FLOAT;
    if (v->tex && !v->store_released && (sampler == VR_SAMPLER_MANUAL || vr_tex_texel(v->tex) != texel)) {
        /* the arrays of the other texel width, or arrays nobody uses any more: their memory goes back */
        VR_CUDA(v, cudaDeviceSynchronize());
        vr_tex_destroy(v->tex);
        v->tex = NULL;
        v->tex_valid = false;
    }
    if (sampler != VR_SAMPLER_MANUAL && !v->tex) {
        const VrGrid& g = v->grid;
        if (!(g.layout == VR_LAYOUT_TILED && g.tl[0] == 2 && g.tl[1] == 2 && g.tl[2] == 1 && g.ml[0] == 0 && g.ml[1] == 0 && g.ml[2] == 0))
            return fail(v, VR_ERR_STATE, "vr_set_sampler: the texture arm is built beside the default (4x4x2 tiled) store only");
        /* ask first: creating ~100 arrays until one fails and freeing them again takes seconds and has been seen to leave the
         * process with slow host copies afterwards (bench.py --sharding bricks on the 103 GB cube) */
        size_t free_b = 0, total_b = 0;
        const double need_b = (double)g.slot * g.nown * (texel == VR_TEXEL_FLOAT ? 4.0 : texel == VR_TEXEL_HALF ? 2.0 : 1.0);
        cudaError_t e = cudaMemGetInfo(&free_b, &total_b);
        if (e == cudaSuccess && (double)free_b < need_b * 1.01 + 64e6) e = cudaErrorMemoryAllocation;
        if (e == cudaSuccess) e = vr_tex_create(g, &v->tex, true, texel);
        if (e != cudaSuccess) v->sampler = VR_SAMPLER_MANUAL; /* no arrays (any of another width were freed above): hand-rolled */
        if (e != cudaSuccess)
            return fail(v, e == cudaErrorMemoryAllocation ? VR_ERR_OUT_OF_MEMORY : VR_ERR_CUDA,
                        "vr_set_sampler: 3-D arrays for %d bricks (%.2f GB beside the brick store): %s", g.nown,
                        (double)g.slot * g.nown * (texel == VR_TEXEL_FLOAT ? 4.0 : texel == VR_TEXEL_HALF ? 2.0 : 1.0) / 1e9, cudaGetErrorString(e));
        v->tex_valid = false;
    }
    v->sampler = sampler;
    return VR_OK;
}

/* texture arm: bring the arrays up to date with the store (one launch, after an upload only) */
static int ensure_tex(vr_volume* v, cudaStream_t st) {
    if (v->tex_valid) return VR_OK;
    if (vr_tex_texel(v->tex) == VR_TEXEL_BYTE) { /* byte texels are scaled with the bricks' ranges (row f1) */
        const int rc = ensure_minmax(v, st);
        if (rc) return rc;
    }
    VR_CUDA(v, vr_launch_tex_fill(v->grid, v->bricks, v->tex, v->d_mm, st));
    v->launches++;
    v->tex_valid = true;
    return VR_OK;
}

extern "C" int vr_volume_release_store(vr_volume* v, int64_t* freed_bytes_out, void* stream) {
    if (!v) return fail(NULL, VR_ERR_INVALID_ARG, "vr_volume_release_store: NULL handle");
    if (freed_bytes_out) *freed_bytes_out = 0;
    if (!v->vmm) return fail(v, VR_ERR_STATE, "vr_volume_release_store: the handle was not created with VR_LAYOUT_TILED_RELEASABLE");
    if (!v->has_data) return fail(v, VR_ERR_STATE, "vr_volume_release_store: nothing uploaded");
    if (v->store_released) return fail(v, VR_ERR_STATE, "vr_volume_release_store: already released");
    cudaStream_t st = (cudaStream_t)stream;
    int rc = ensure_minmax(v, st); /* the range tables (rows f1, R19) are read from the store: last chance */
    if (rc) return rc;
    VR_CUDA(v, cudaDeviceSynchronize());
    if (v->tex) { /* a second copy made by vr_set_sampler: start over, array by array */
        vr_tex_destroy(v->tex);
        v->tex = NULL;
    }
    const bool to_half = v->sampler == VR_SAMPLER_TEXTURE_HALF; /* the arrays take the texel width of the sampler in force */
    cudaError_t e = vr_tex_create(v->grid, &v->tex, false, to_half ? VR_TEXEL_HALF : VR_TEXEL_FLOAT);
    if (e != cudaSuccess) return fail(v, e == cudaErrorMemoryAllocation ? VR_ERR_OUT_OF_MEMORY : VR_ERR_CUDA, "vr_volume_release_store: %s", cudaGetErrorString(e));
    long long freed = 0;
    for (int s = 0; s < v->grid.nown; ++s) {
        int has_nan = 0;
        e = vr_tex_convert_slot(v->grid, v->bricks, v->tex, s, &has_nan, st);
        v->launches++;
        if (e != cudaSuccess) {
            cudaGetLastError();
            /* the slots converted so far are gone from the store: the handle can only be destroyed */
            v->store_released = true;
            v->has_data = false;
            return fail(v, e == cudaErrorMemoryAllocation ? VR_ERR_OUT_OF_MEMORY : VR_ERR_CUDA,
                        "vr_volume_release_store: slot %d of %d: %s (the handle is no longer usable)", s, v->grid.nown, cudaGetErrorString(e));
        }
        if (!has_nan) freed += (long long)vr_vmm_release_slot(v->vmm, s); /* R14 needs the float32 cells of blanked bricks */
    }
    v->store_released = true;
    v->tex_valid = true;
    v->sampler = to_half ? VR_SAMPLER_TEXTURE_HALF : VR_SAMPLER_TEXTURE;
    if (freed_bytes_out) *freed_bytes_out = freed;
    return VR_OK;
}

extern "C" int vr_set_culling(vr_volume* v, int enable) {
    if (!v) return fail(NULL, VR_ERR_INVALID_ARG, "vr_set_culling: NULL handle");
    v->culling = enable != 0;
    return VR_OK;
}

extern "C" int vr_debug_cell_flags(vr_volume* v, int b, unsigned char* flags_out, int* dims) {
    if (!v) return fail(NULL, VR_ERR_INVALID_ARG, "vr_debug_cell_flags: NULL handle");
    if (!dims || b < 0 || b >= v->grid.nbricks) return fail(v, VR_ERR_INVALID_ARG, "vr_debug_cell_flags: bad brick %d or NULL dims", b);
    const int slot_b = vr_slot_index(v->grid, b);
    if (slot_b < 0) return fail(v, VR_ERR_INVALID_ARG, "vr_debug_cell_flags: this part does not hold brick %d", b);
    if (!v->has_data || !v->has_tf) return fail(v, VR_ERR_STATE, "vr_debug_cell_flags: needs data and a transfer function");
    if (!cells_supported(v)) return fail(v, VR_ERR_STATE, "vr_debug_cell_flags: macro-cells need the 4x4x2 layout and ghost >= 1");
    const int rc = ensure_cells(v, true, 0);
    if (rc) return rc;
    for (int a = 0; a < 3; ++a) dims[a] = v->nc[a];
    if (!flags_out) return VR_OK;
    VR_CUDA(v, cudaDeviceSynchronize());
    unsigned* words = new (std::nothrow) unsigned[v->cell_words];
    if (!words) return fail(v, VR_ERR_OUT_OF_MEMORY, "vr_debug_cell_flags: host allocation failed");
    const cudaError_t e = cudaMemcpy(words, v->d_cell_bits + (size_t)slot_b * v->cell_words, sizeof(unsigned) * v->cell_words,
                                     cudaMemcpyDeviceToHost);
    if (e == cudaSuccess)
        for (int m = 0; m < v->nc[0] * v->nc[1] * v->nc[2]; ++m) flags_out[m] = (unsigned char)((words[m >> 5] >> (m & 31)) & 1u);
    delete[] words;
    VR_CUDA(v, e);
    return VR_OK;
}

/* R23: measured error of the texture arm's filtered fetch in brick b (test / measurement export) */
extern "C" int vr_debug_tex_error(vr_volume* v, int b, int64_t n, unsigned seed, float* max_err_out, float* range_out) {
    if (!v) return fail(NULL, VR_ERR_INVALID_ARG, "vr_debug_tex_error: NULL handle");
    if (!max_err_out || !range_out || n < 1 || b < 0 || b >= v->grid.nbricks) return fail(v, VR_ERR_INVALID_ARG, "vr_debug_tex_error: bad argument");
    const int slot_b = vr_slot_index(v->grid, b);
    if (slot_b < 0) return fail(v, VR_ERR_INVALID_ARG, "vr_debug_tex_error: this part does not hold brick %d", b);
    if (!v->has_data || v->store_released || v->sampler == VR_SAMPLER_MANUAL || !v->tex)
        return fail(v, VR_ERR_STATE, "vr_debug_tex_error: needs data, a texture sampler and the float32 store");
    int rc = ensure_minmax(v, 0);
    if (!rc) rc = ensure_tex(v, 0);
    if (rc) return rc;
    float2 mm;
    VR_CUDA(v, cudaMemcpy(&mm, v->d_mm + b, sizeof(mm), cudaMemcpyDeviceToHost));
    const bool byte = vr_tex_texel(v->tex) == VR_TEXEL_BYTE;
    float* d_err = NULL;
    VR_CUDA(v, cudaMalloc(&d_err, sizeof(float)));
    cudaError_t e = cudaMemset(d_err, 0, sizeof(float));
    if (e == cudaSuccess) e = vr_launch_tex_error(v->grid, v->bricks, v->tex, slot_b, n, seed, byte ? mm.y - mm.x : 1.0f, byte ? mm.x : 0.0f, d_err, 0);
    if (e == cudaSuccess) e = cudaMemcpy(max_err_out, d_err, sizeof(float), cudaMemcpyDeviceToHost);
    cudaFree(d_err);
    VR_CUDA(v, e);
    v->launches++;
    *range_out = mm.y - mm.x;
    return VR_OK;
}

/* R20 (vii): the quantities the texture arm's ALPHA guard is decided on (test / measurement export) */
extern "C" int vr_debug_tex_alpha_guard(vr_volume* v, float* mean_cell_range_out, float* table_slope_out, int* ok_out) {
    if (!v) return fail(NULL, VR_ERR_INVALID_ARG, "vr_debug_tex_alpha_guard: NULL handle");
    if (!mean_cell_range_out || !table_slope_out || !ok_out) return fail(v, VR_ERR_INVALID_ARG, "vr_debug_tex_alpha_guard: NULL output");
    if (!v->has_data || !v->has_tf) return fail(v, VR_ERR_STATE, "vr_debug_tex_alpha_guard: needs data and a transfer function");
    const int rc = decide_tex_alpha(v, 0);
    if (rc) return rc;
    *mean_cell_range_out = v->mean_cell_range;
    *table_slope_out = v->tf_slope;
    *ok_out = v->tex_alpha_ok ? 1 : 0;
    return VR_OK;
}

extern "C" int vr_debug_brick_minmax(vr_volume* v, float* mm_out) {
    if (!v) return fail(NULL, VR_ERR_INVALID_ARG, "vr_debug_brick_minmax: NULL handle");
    if (!mm_out) return fail(v, VR_ERR_INVALID_ARG, "vr_debug_brick_minmax: NULL output");
    if (!v->has_data) return fail(v, VR_ERR_STATE, "vr_debug_brick_minmax: nothing uploaded");
    const int rc = ensure_minmax(v, 0);
    if (rc) return rc;
    VR_CUDA(v, cudaDeviceSynchronize());
    VR_CUDA(v, cudaMemcpy(mm_out, v->d_mm, sizeof(float2) * v->grid.nbricks, cudaMemcpyDeviceToHost));
    return VR_OK;
}

/* pieces: the frame leaves as n windows (x0, y0, x1, y1), window q stored [y1-y0][x1-x0] at ptrs[q] (row f3) */
struct VrPieces {
    int n;
    const int* rects;
    float* const* ptrs;
};

static int render_frame(vr_volume* v, const float* view, const float* proj, int width, int height, float step, int mode,
                        float* out_rgba, void* stream, bool partial, const VrPieces* pieces);

extern "C" int vr_render(vr_volume* v, const float* view, const float* proj, int width, int height, float step, int mode,
                         float* out_rgba, void* stream) {
    return render_frame(v, view, proj, width, height, step, mode, out_rgba, stream, false, NULL);
}

extern "C" int vr_render_part(vr_volume* v, const float* view, const float* proj, int width, int height, float step, int mode,
                              float* out_part, int* rect_out, void* stream) {
    const int rc = render_frame(v, view, proj, width, height, step, mode, out_part, stream, true, NULL);
    if (rc) return rc;
    if (rect_out && vr_host_part_rect(v->grid, view, proj, width, height, rect_out))
        return fail(v, VR_ERR_INVALID_ARG, "vr_render_part: proj*view is singular");
    return VR_OK;
}

extern "C" int vr_render_part_pieces(vr_volume* v, const float* view, const float* proj, int width, int height, float step,
                                     int mode, const int* piece_rects, float* const* pieces, int npieces, void* stream) {
    if (!v) return fail(NULL, VR_ERR_INVALID_ARG, "vr_render_part_pieces: NULL handle");
    if (npieces < 0 || npieces > 4096 || (npieces > 0 && (!piece_rects || !pieces)))
        return fail(v, VR_ERR_INVALID_ARG, "vr_render_part_pieces: bad piece list");
    if (v->traversal != VR_SORT_LAST) return fail(v, VR_ERR_STATE, "vr_render_part_pieces: needs the VR_SORT_LAST traversal");
    for (int q = 0; q < npieces; ++q) {
        const int* r = piece_rects + 4 * q;
        if (r[0] < 0 || r[1] < 0 || r[2] > width || r[3] > height || r[2] < r[0] || r[3] < r[1])
            return fail(v, VR_ERR_INVALID_ARG, "vr_render_part_pieces: piece %d leaves the %dx%d frame", q, width, height);
        if (!pieces[q] && r[2] > r[0] && r[3] > r[1]) return fail(v, VR_ERR_INVALID_ARG, "vr_render_part_pieces: piece %d is NULL", q);
    }
    const VrPieces pc = {npieces, piece_rects, pieces};
    float dummy; /* render_frame wants a non-NULL output; with pieces it is not written */
    return render_frame(v, view, proj, width, height, step, mode, &dummy, stream, true, &pc);
}

extern "C" int vr_part_rect(int nx, int ny, int nz, int brick, const int* b0, const int* b1, const float* view, const float* proj,
                            int width, int height, int* rect_out) {
    if (!b0 || !b1 || !view || !proj || !rect_out) return fail(NULL, VR_ERR_INVALID_ARG, "vr_part_rect: NULL argument");
    if (nx <= 0 || ny <= 0 || nz <= 0 || brick < 2 || width <= 0 || height <= 0)
        return fail(NULL, VR_ERR_INVALID_ARG, "vr_part_rect: bad volume, brick or frame size");
    VrGrid g;
    memset(&g, 0, sizeof(g));
    g.n[0] = nx; g.n[1] = ny; g.n[2] = nz;
    g.brick = brick;
    g.part = 1;
    long long nb = 1;
    for (int a = 0; a < 3; ++a) {
        g.g[a] = (g.n[a] + brick - 1) / brick;
        nb *= g.g[a];
        if (b0[a] < 0 || b1[a] <= b0[a] || b1[a] > g.g[a]) return fail(NULL, VR_ERR_INVALID_ARG, "vr_part_rect: bad brick box");
        g.pb0[a] = b0[a], g.pb1[a] = b1[a];
    }
    if (nb > 65535) return fail(NULL, VR_ERR_INVALID_ARG, "vr_part_rect: %lld bricks > 65535", nb);
    g.nbricks = (int)nb;
    if (vr_host_part_rect(g, view, proj, width, height, rect_out)) return fail(NULL, VR_ERR_INVALID_ARG, "vr_part_rect: proj*view is singular");
    return VR_OK;
}

extern "C" int vr_kd_partition(int nx, int ny, int nz, int brick, int nparts, int* boxes_out, int* tree_out) {
    if (!boxes_out || !tree_out) return fail(NULL, VR_ERR_INVALID_ARG, "vr_kd_partition: NULL output");
    if (nx <= 0 || ny <= 0 || nz <= 0 || brick < 2) return fail(NULL, VR_ERR_INVALID_ARG, "vr_kd_partition: bad volume or brick size");
    long long nb = 1;
    for (int a = 0; a < 3; ++a) nb *= ((a == 0 ? nx : a == 1 ? ny : nz) + brick - 1) / brick;
    if (nparts < 1 || nparts > nb || nb > 65535)
        return fail(NULL, VR_ERR_INVALID_ARG, "vr_kd_partition: %d parts for %lld bricks", nparts, nb);
    if (vr_host_kd_partition(nx, ny, nz, brick, nparts, boxes_out, tree_out))
        return fail(NULL, VR_ERR_INVALID_ARG, "vr_kd_partition: the brick grid cannot be cut into %d boxes this way", nparts);
    return VR_OK;
}

extern "C" int vr_part_order(const int* tree, int nparts, int brick, const float* view, const float* proj, int* order_out) {
    if (!tree || !view || !proj || !order_out || nparts < 1 || brick < 2)
        return fail(NULL, VR_ERR_INVALID_ARG, "vr_part_order: NULL or bad argument");
    const int rc = vr_host_part_order(tree, nparts, brick, view, proj, order_out);
    if (rc == 1) return fail(NULL, VR_ERR_INVALID_ARG, "vr_part_order: proj*view is singular");
    if (rc) return fail(NULL, VR_ERR_INVALID_ARG, "vr_part_order: malformed tree");
    return VR_OK;
}

/* partial: the frame is one part's contribution to a sort-last frame (row f3): a MIP frame stays scalar */
static int render_frame(vr_volume* v, const float* view, const float* proj, int width, int height, float step, int mode,
                        float* out_rgba, void* stream, bool partial, const VrPieces* pieces) {
    long long sub_px = 0, items = 0;
    int rc = check_view(v, "vr_render", view, proj, width, height, &sub_px, &items);
    if (rc) return rc;
    rc = check_overflow(v, "vr_render");
    if (rc) return rc;
    if (partial && mode == VR_MIP && v->traversal == VR_FUSED)
        return fail(v, VR_ERR_STATE, "vr_render_part: VR_MIP parts need the VR_SORT_LAST traversal");
    if (!out_rgba) return fail(v, VR_ERR_INVALID_ARG, "vr_render: NULL output");
    if (!(step >= 0.0f) || !isfinite(step)) return fail(v, VR_ERR_INVALID_ARG, "vr_render: step must be > 0, or VR_STEP_AUTO (0)");
    if (mode != VR_ALPHA && mode != VR_MIP) return fail(v, VR_ERR_INVALID_ARG, "vr_render: bad mode %d", mode);
    if (!v->has_tf) return fail(v, VR_ERR_STATE, "vr_render: no transfer function set");
    if (!v->has_data) return fail(v, VR_ERR_STATE, "vr_render: nothing uploaded");
    if (v->store_released) {
        if (mode != VR_ALPHA) return fail(v, VR_ERR_STATE, "vr_render: VR_MIP needs the float32 store, which was released");
        if (!v->tf_smooth) return fail(v, VR_ERR_STATE, "vr_render: a transfer function with a step needs the float32 store, which was released");
        if (v->counting == 2) return fail(v, VR_ERR_STATE, "vr_render: counting mode 2 needs the float32 store, which was released");
        if (!(step >= 0.9f && step <= 1.0f))
            return fail(v, VR_ERR_STATE, "vr_render: on a released store the step must lie in [0.9, 1] voxels (the opacity correction multiplies "
                                         "the texture filter's error by the step, and for smaller steps without bound where the table's "
                                         "opacity nears 1: such frames need the float32 store, DESIGN.md R20)");
    }
    rc = ensure_sub(v, sub_px);
    if (rc) return rc;
    if (v->traversal == VR_SORT_LAST) {
        rc = ensure_rays(v, (long long)width * height);
        if (rc) return rc;
    }
    cudaStream_t st = (cudaStream_t)stream;
    const bool timing = v->timing;
    cudaEvent_t* ev = v->ev[v->timed_frames % VR_EV_RING];

    if (v->culling) { /* after an upload only: the range pass is not part of the frame's stages */
        rc = ensure_minmax(v, st);
        if (rc) return rc;
    }
    /* after an upload or a new transfer function only, and only if the table has a transparent range */
    const bool skipping = v->culling && v->tf_has_zero && mode == VR_ALPHA && cells_supported(v);
    if (skipping) {
        rc = ensure_cells(v, true, st);
        if (rc) return rc;
    }
    bool mip_skipping = false;
    if (v->culling && mode == VR_MIP && cells_supported(v)) {
        rc = decide_mip_skip(v, st);
        if (rc) return rc;
        mip_skipping = v->mip_skip_useful;
    }
    /* texture arm: ALPHA frames with a smooth table take their values from the arrays; MIP frames use the arrays as an exact
     * filter in front of the hand-rolled sampler (needs the float32 store and the bricks' ranges; where stepping over empty
     * macro-cells pays, that stays) */
    /* R20: the opacity correction 1 - (1 - a)^w multiplies the filter's per-sample error by the step w: ALPHA values come from the
     * arrays for steps up to one voxel only (the randomised suite found 2.2e-3 at step 1.63; VR_STEP_AUTO's per-ray steps are >= 1) */
    bool tex_alpha = (v->sampler == VR_SAMPLER_TEXTURE || v->sampler == VR_SAMPLER_TEXTURE_HALF) && mode == VR_ALPHA && v->counting != 2 && v->tf_smooth &&
                     step > 0.0f && step <= 1.0f;
    if (tex_alpha) { /* R20 (vii): only while the data's voxel-to-voxel differences are small enough against this table */
        rc = decide_tex_alpha(v, st);
        if (rc) return rc;
        if (!v->tex_alpha_ok) {
            if (v->store_released)
                return fail(v, VR_ERR_STATE, "vr_render: the texture filter is too coarse for this data under this transfer function (mean macro-cell "
                                             "range %g against a table range of %g, table slope %g: DESIGN.md R20) and the float32 store was released",
                            (double)v->mean_cell_range, (double)(v->lut.vmax - v->lut.vmin), (double)v->tf_slope);
            tex_alpha = false; /* the hand-rolled sampler */
        }
    }
    if (tex_alpha && v->sampler == VR_SAMPLER_TEXTURE_HALF) { /* R22: only while float16 is fine enough for this data under this table */
        rc = decide_half_alpha(v, st);
        if (rc) return rc;
        if (!v->half_alpha_ok) {
            if (v->store_released)
                return fail(v, VR_ERR_STATE, "vr_render: float16 texels are too coarse for this data under this transfer function (largest "
                                             "magnitude / 1024 > 1.5e-3 of the table's range) and the float32 store was released");
            tex_alpha = false; /* the hand-rolled sampler */
        }
    }
    const bool tex_mip = v->sampler != VR_SAMPLER_MANUAL && mode == VR_MIP && v->counting != 2 && !v->store_released &&
                         v->traversal == VR_SORT_LAST && !mip_skipping;
    const bool use_tex = tex_alpha || tex_mip;
    if (use_tex) { /* after an upload only */
        rc = ensure_tex(v, st);
        if (rc) return rc;
    }
    if (tex_mip) {
        rc = ensure_minmax(v, st);
        if (rc) return rc;
    }
    if (timing) VR_CUDA(v, cudaEventRecord(ev[0], st));
    rc = run_setup(v, view, proj, width, height, mode, v->culling, st);
    if (rc) return rc;
    /* brick faces of brick^2 voxels project onto sub_px pixels in all: > 4 voxels per pixel = sparse */
    const bool sparse = (double)v->grid.nown * v->grid.brick * v->grid.brick > 4.0 * (double)sub_px;
    const bool ray_table = v->traversal == VR_SORT_LAST && !sparse;
    if (ray_table) { /* the per-ray part of row a4, once per pixel: part of the set-up stage (dense views only) */
        VR_CUDA(v, vr_launch_rays(v->grid, v->d_vs, width, height, (double)step, v->d_rays, st));
        v->launches++;
    }
    if (timing) VR_CUDA(v, cudaEventRecord(ev[1], st));

    VrRaycastParams p;
    p.grid = v->grid;
    p.bricks = v->bricks;
    p.rays = ray_table ? v->d_rays : NULL;
    p.ray_plane = (long long)width * height;
    p.vs = v->d_vs;
    p.bv = v->d_bv;
    p.order = v->d_order;
    p.item_prefix = v->d_item_prefix;
    p.vs_rw = v->d_vs;
    p.sub = v->d_sub;
    p.bitmap = NULL;
    p.tex = use_tex ? vr_tex_table(v->tex) : NULL;
    p.tex_nan = use_tex ? vr_tex_nan_table(v->tex) : NULL;
    p.brick_mm = tex_mip ? v->d_mm : NULL;
    /* R20's guard: with steps below one voxel the opacity correction (1 - a)^w has an unbounded slope where the table's opacity nears
     * 1, so such samples are re-evaluated by the hand-rolled sampler (needs the float32 store: checked above for a released one) */
    p.tex_guard = (tex_alpha && !v->store_released && step < 1.0f) ? 0.9f : 2.0f;
    p.tex_only = v->store_released ? 1 : 0;
    const int texel = tex_mip ? vr_tex_texel(v->tex) : VR_TEXEL_FLOAT;
    p.mip_range_eps = 1.0f / 64.0f + (texel == VR_TEXEL_BYTE ? 1.0f / 500.0f : 0.0f); /* half a byte step is range / 510 */
    p.mip_mag_eps = texel == VR_TEXEL_HALF ? 1.0f / 512.0f : texel == VR_TEXEL_BYTE ? 1.0f / 4096.0f : 1.0f / 16384.0f;
    p.mip_mag_max = texel == VR_TEXEL_HALF ? 60000.0f : INFINITY;
    p.mip_abs_eps = texel == VR_TEXEL_HALF ? 1.1920929e-7f /* 2^-23: four half-steps of float16's subnormal grid */ : 2.4e-38f;
    p.tex_byte = texel == VR_TEXEL_BYTE;
    p.cell_bits = skipping ? v->d_cell_bits : NULL;
    p.cell_mm = mip_skipping ? v->d_cell_mm : NULL;
    p.nc[0] = v->nc[0]; p.nc[1] = v->nc[1]; p.nc[2] = v->nc[2];
    p.cell_words = v->cell_words;
    if (v->counting == 2) {
        VR_CUDA(v, cudaMemsetAsync(v->d_bitmap, 0, (size_t)v->bitmap_words * sizeof(unsigned), st));
        p.bitmap = v->d_bitmap;
    }
    p.lut = v->lut;
    p.step = (double)step;
    p.tau = v->tau;
    p.mode = mode;
    if (v->traversal == VR_FUSED) {
        VR_CUDA(v, vr_launch_fused(p, out_rgba, width, height, v->counting != 0, st));
        v->launches++;
        if (timing) VR_CUDA(v, cudaEventRecord(ev[2], st));
    } else {
        VR_CUDA(v, vr_launch_raycast(p, items, v->counting != 0, sparse, st));
        v->launches++;
        if (timing) VR_CUDA(v, cudaEventRecord(ev[2], st));
        const int kmode = (partial && mode == VR_MIP) ? VR_MIP_RAW : mode;
        if (!pieces) {
            VR_CUDA(v, vr_launch_composite(v->d_layers, v->d_order, v->grid.nbricks, width, height, kmode, v->lut, out_rgba,
                                           v->d_vs->bound, NULL, st));
            v->launches++;
        }
        /* stage-1 compositing straight into the rectangle-packed pieces the part sends */
        for (int q = 0; pieces && q < pieces->n; ++q) {
            const int* r = pieces->rects + 4 * q;
            if (r[2] <= r[0] || r[3] <= r[1]) continue;
            VR_CUDA(v, vr_launch_composite(v->d_layers, v->d_order, v->grid.nbricks, width, height, kmode, v->lut, pieces->ptrs[q],
                                           v->d_vs->bound, r, st));
            v->launches++;
        }
    }
    if (timing) {
        VR_CUDA(v, cudaEventRecord(ev[3], st));
        v->timed_frames++;
    }
    v->last_W = width;
    v->last_H = height;
    v->last_mode = mode;
    v->last_valid = v->traversal == VR_SORT_LAST; /* fused frames leave no sub-images to inspect */
    v->last_stats_valid = true;
    return VR_OK;
}

extern "C" int vr_render_host(vr_volume* v, const float* view, const float* proj, int width, int height, float step, int mode,
                              float* out_rgba_host, void* stream) {
    if (!v) return fail(NULL, VR_ERR_INVALID_ARG, "vr_render_host: NULL handle");
    if (!out_rgba_host) return fail(v, VR_ERR_INVALID_ARG, "vr_render_host: NULL output");
    if (width <= 0 || height <= 0 || width > 32768 || height > 32768)
        return fail(v, VR_ERR_INVALID_ARG, "vr_render_host: bad frame size %dx%d", width, height);
    const long long px = (long long)width * height;
    if (px > v->frame_capacity_px) {
        if (v->d_frame) {
            VR_CUDA(v, cudaDeviceSynchronize());
            v_free(v, v->d_frame); /* only the synchronous entry's own frame: the pipelined entry's frames, events and stream stay */
            v->d_frame = NULL;
            v->frame_capacity_px = 0;
        }
        VR_CUDA(v, v_alloc(v, &v->d_frame, (size_t)px * 16));
        v->frame_capacity_px = px;
    }
    const int rc = vr_render(v, view, proj, width, height, step, mode, v->d_frame, stream);
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    VR_CUDA(v, cudaMemcpyAsync(out_rgba_host, v->d_frame, (size_t)px * 16, cudaMemcpyDeviceToHost, st));
    VR_CUDA(v, cudaStreamSynchronize(st));
    return check_overflow(v, "vr_render_host");
}

extern "C" int vr_render_host_async(vr_volume* v, const float* view, const float* proj, int width, int height, float step,
                                    int mode, float* out_rgba_host, void* stream) {
    if (!v) return fail(NULL, VR_ERR_INVALID_ARG, "vr_render_host_async: NULL handle");
    if (!out_rgba_host) return fail(v, VR_ERR_INVALID_ARG, "vr_render_host_async: NULL output");
    if (width <= 0 || height <= 0 || width > 32768 || height > 32768)
        return fail(v, VR_ERR_INVALID_ARG, "vr_render_host_async: bad frame size %dx%d", width, height);
    const long long px = (long long)width * height;
    const int rcp = ensure_pipe(v, px);
    if (rcp) return rcp;
    cudaStream_t st = (cudaStream_t)stream;
    const int slot = (int)(v->pipe_frames & 1);
    /* the frame that last used this slot must have left it */
    if (v->pipe_frames >= 2) VR_CUDA(v, cudaStreamWaitEvent(st, v->ev_copied[slot], 0));
    const int rc = vr_render(v, view, proj, width, height, step, mode, v->d_pipe[slot], stream);
    if (rc) return rc;
    VR_CUDA(v, cudaEventRecord(v->ev_rendered[slot], st));
    VR_CUDA(v, cudaStreamWaitEvent(v->copy_stream, v->ev_rendered[slot], 0));
    VR_CUDA(v, cudaMemcpyAsync(out_rgba_host, v->d_pipe[slot], (size_t)px * 16, cudaMemcpyDeviceToHost, v->copy_stream));
    VR_CUDA(v, cudaEventRecord(v->ev_copied[slot], v->copy_stream));
    v->pipe_frames++;
    return VR_OK;
}

extern "C" int vr_render_host_wait(vr_volume* v) {
    if (!v) return fail(NULL, VR_ERR_INVALID_ARG, "vr_render_host_wait: NULL handle");
    if (v->copy_stream) VR_CUDA(v, cudaStreamSynchronize(v->copy_stream));
    return check_overflow(v, "vr_render_host_wait");
}

/* ------------------------------------------------------------------------------------------ */
static int composite_layers(const VrLut& lut, int kmode, const float* const* layers, const int* rects, const int* order, int n,
                            int width, int height, float* out, void* stream);

extern "C" int vr_composite(const float* const* layers, const int* rects, const int* order, int n, int width, int height,
                            float* out, void* stream) {
    VrLut none;
    memset(&none, 0, sizeof(none));
    return composite_layers(none, VR_ALPHA, layers, rects, order, n, width, height, out, stream);
}

extern "C" int vr_composite_parts(vr_volume* v, int mode, const float* const* parts, const int* rects, const int* order, int n,
                                  int width, int height, float* out, void* stream) {
    if (!v) return fail(NULL, VR_ERR_INVALID_ARG, "vr_composite_parts: NULL handle");
    if (mode != VR_ALPHA && mode != VR_MIP) return fail(v, VR_ERR_INVALID_ARG, "vr_composite_parts: bad mode %d", mode);
    if (mode == VR_MIP && !v->has_tf) return fail(v, VR_ERR_STATE, "vr_composite_parts: no transfer function set");
    const int rc = composite_layers(v->lut, mode == VR_MIP ? VR_MIP_PARTS : VR_ALPHA, parts, rects, order, n, width, height, out, stream);
    if (rc == VR_OK) v->launches++;
    return rc;
}

static int composite_layers(const VrLut& lut, int kmode, const float* const* layers, const int* rects, const int* order, int n,
                            int width, int height, float* out, void* stream) {
    if (!layers || !rects || !order || !out) return fail(NULL, VR_ERR_INVALID_ARG, "vr_composite: NULL argument");
    if (n < 0 || n > 4096) return fail(NULL, VR_ERR_INVALID_ARG, "vr_composite: n = %d outside [0,4096]", n);
    if (width <= 0 || height <= 0 || width > 32768 || height > 32768)
        return fail(NULL, VR_ERR_INVALID_ARG, "vr_composite: bad frame size %dx%d", width, height);
    VrCompLayer* tab = new (std::nothrow) VrCompLayer[n > 0 ? n : 1];
    unsigned char* seen = new (std::nothrow) unsigned char[n > 0 ? n : 1];
    if (!tab || !seen) {
        delete[] tab;
        delete[] seen;
        return fail(NULL, VR_ERR_OUT_OF_MEMORY, "vr_composite: host allocation failed");
    }
    struct Free { /* released on every return path */
        VrCompLayer* t;
        unsigned char* s;
        ~Free() { delete[] t; delete[] s; }
    } free_tables = {tab, seen};
    memset(seen, 0, (size_t)(n > 0 ? n : 1));
    for (int l = 0; l < n; ++l) {
        const int* r = rects + 4 * l;
        if (r[0] < 0 || r[1] < 0 || r[2] > width || r[3] > height || r[2] < r[0] || r[3] < r[1])
            return fail(NULL, VR_ERR_INVALID_ARG, "vr_composite: rectangle %d outside the viewport", l);
        if (!layers[l] && r[2] > r[0] && r[3] > r[1]) return fail(NULL, VR_ERR_INVALID_ARG, "vr_composite: layer %d is NULL", l);
        if (order[l] < 0 || order[l] >= n || seen[order[l]]) return fail(NULL, VR_ERR_INVALID_ARG, "vr_composite: order is not a permutation");
        seen[order[l]] = 1;
        VrCompLayer& L = tab[l];
        L.x0 = r[0]; L.y0 = r[1]; L.x1 = r[2]; L.y1 = r[3];
        L.sx0 = r[0]; L.sy0 = r[1];
        L.pitch = r[2] - r[0];
        L.pad = 0;
        L.addr = (unsigned long long)(uintptr_t)layers[l];
    }
    cudaStream_t st = (cudaStream_t)stream;
    VrCompLayer* d_tab = NULL;
    int* d_order = NULL;
    const size_t nn = n > 0 ? (size_t)n : 1;
    VR_CUDA(NULL, cudaMallocAsync(&d_tab, sizeof(VrCompLayer) * nn, st));
    VR_CUDA(NULL, cudaMallocAsync(&d_order, sizeof(int) * nn, st));
    if (n > 0) {
        VR_CUDA(NULL, cudaMemcpyAsync(d_tab, tab, sizeof(VrCompLayer) * n, cudaMemcpyHostToDevice, st));
        VR_CUDA(NULL, cudaMemcpyAsync(d_order, order, sizeof(int) * n, cudaMemcpyHostToDevice, st));
    }
    VR_CUDA(NULL, vr_launch_composite(d_tab, d_order, n, width, height, kmode, lut, out, NULL, NULL, st));
    VR_CUDA(NULL, cudaFreeAsync(d_tab, st));
    VR_CUDA(NULL, cudaFreeAsync(d_order, st));
    return VR_OK;
}

/* ------------------------------------------------------------------------------------------
 * Debug / test exports. They run the same set-up kernel a frame runs and read its tables.
 * ---------------------------------------------------------------------------------------- */
static int debug_setup(vr_volume* v, const char* who, const float* view, const float* proj, int W, int H) {
    long long sub_px = 0, items = 0;
    int rc = check_view(v, who, view, proj, W, H, &sub_px, &items);
    if (rc) return rc;
    rc = ensure_sub(v, sub_px);
    if (rc) return rc;
    rc = run_setup(v, view, proj, W, H, VR_ALPHA, false, 0);
    if (rc) return rc;
    v->last_valid = false; /* the sub-image offsets of the last frame are gone */
    v->last_stats_valid = false;
    VR_CUDA(v, cudaDeviceSynchronize());
    return VR_OK;
}

extern "C" int vr_debug_brick_order(vr_volume* v, const float* view, const float* proj, int* order_out) {
    if (v && !order_out) return fail(v, VR_ERR_INVALID_ARG, "vr_debug_brick_order: NULL output");
    const int rc = debug_setup(v, "vr_debug_brick_order", view, proj, 16, 16);
    if (rc) return rc;
    VR_CUDA(v, cudaMemcpy(order_out, v->d_order, sizeof(int) * v->grid.nbricks, cudaMemcpyDeviceToHost));
    return VR_OK;
}

extern "C" int vr_debug_rects(vr_volume* v, const float* view, const float* proj, int width, int height, int* rects_out) {
    if (v && !rects_out) return fail(v, VR_ERR_INVALID_ARG, "vr_debug_rects: NULL output");
    const int rc = debug_setup(v, "vr_debug_rects", view, proj, width, height);
    if (rc) return rc;
    const int nb = v->grid.nbricks;
    VrBrickView* h = new (std::nothrow) VrBrickView[nb];
    if (!h) return fail(v, VR_ERR_OUT_OF_MEMORY, "vr_debug_rects: host allocation failed");
    cudaError_t e = cudaMemcpy(h, v->d_bv, sizeof(VrBrickView) * nb, cudaMemcpyDeviceToHost);
    if (e == cudaSuccess)
        for (int b = 0; b < nb; ++b) {
            rects_out[4 * b + 0] = h[b].rx0;
            rects_out[4 * b + 1] = h[b].ry0;
            rects_out[4 * b + 2] = h[b].rx1;
            rects_out[4 * b + 3] = h[b].ry1;
        }
    delete[] h;
    VR_CUDA(v, e);
    return VR_OK;
}

extern "C" int vr_debug_ray_bricks(vr_volume* v, const float* view, const float* proj, int width, int height,
                                   const int* pixels, int npix, int* counts, int* lists, int maxlen, uint8_t* grazing) {
    if (v && (!pixels || !counts || !lists || npix <= 0 || maxlen <= 0))
        return fail(v, VR_ERR_INVALID_ARG, "vr_debug_ray_bricks: NULL or empty argument");
    int rc = debug_setup(v, "vr_debug_ray_bricks", view, proj, width, height);
    if (rc) return rc;
    int *d_pix = NULL, *d_counts = NULL, *d_lists = NULL;
    double* d_tins = NULL;
    unsigned char* d_gz = NULL;
    cudaError_t e = cudaMalloc(&d_pix, sizeof(int) * 2 * (size_t)npix);
    if (e == cudaSuccess) e = cudaMalloc(&d_counts, sizeof(int) * (size_t)npix);
    if (e == cudaSuccess) e = cudaMalloc(&d_lists, sizeof(int) * (size_t)npix * maxlen);
    if (e == cudaSuccess) e = cudaMalloc(&d_tins, sizeof(double) * (size_t)npix * maxlen);
    if (e == cudaSuccess) e = cudaMalloc(&d_gz, (size_t)npix);
    if (e == cudaSuccess) e = cudaMemcpy(d_pix, pixels, sizeof(int) * 2 * (size_t)npix, cudaMemcpyHostToDevice);
    if (e == cudaSuccess) {
        e = vr_launch_ray_bricks(v->grid, v->d_vs, d_pix, npix, d_counts, d_lists, d_tins, maxlen, d_gz, 0);
        v->launches++;
    }
    if (e == cudaSuccess) e = cudaDeviceSynchronize();
    if (e == cudaSuccess) e = cudaMemcpy(counts, d_counts, sizeof(int) * (size_t)npix, cudaMemcpyDeviceToHost);
    if (e == cudaSuccess) e = cudaMemcpy(lists, d_lists, sizeof(int) * (size_t)npix * maxlen, cudaMemcpyDeviceToHost);
    if (e == cudaSuccess && grazing) e = cudaMemcpy(grazing, d_gz, (size_t)npix, cudaMemcpyDeviceToHost);
    cudaFree(d_pix);
    cudaFree(d_counts);
    cudaFree(d_lists);
    cudaFree(d_tins);
    cudaFree(d_gz);
    VR_CUDA(v, e);
    return VR_OK;
}

extern "C" int vr_debug_subimages(vr_volume* v, const int* pixels, int npix, float* sub_out) {
    if (!v) return fail(NULL, VR_ERR_INVALID_ARG, "vr_debug_subimages: NULL handle");
    if (!pixels || !sub_out || npix <= 0) return fail(v, VR_ERR_INVALID_ARG, "vr_debug_subimages: NULL or empty argument");
    if (!v->last_valid) return fail(v, VR_ERR_STATE, "vr_debug_subimages: no vr_render since the last debug call");
    for (int q = 0; q < npix; ++q)
        if (pixels[2 * q] < 0 || pixels[2 * q] >= v->last_W || pixels[2 * q + 1] < 0 || pixels[2 * q + 1] >= v->last_H)
            return fail(v, VR_ERR_INVALID_ARG, "vr_debug_subimages: pixel %d outside the last frame", q);
    const int nb = v->grid.nbricks;
    int* d_pix = NULL;
    float* d_out = NULL;
    VR_CUDA(v, cudaDeviceSynchronize());
    cudaError_t e = cudaMalloc(&d_pix, sizeof(int) * 2 * (size_t)npix);
    if (e == cudaSuccess) e = cudaMalloc(&d_out, sizeof(float) * 4 * (size_t)npix * nb);
    if (e == cudaSuccess) e = cudaMemcpy(d_pix, pixels, sizeof(int) * 2 * (size_t)npix, cudaMemcpyHostToDevice);
    if (e == cudaSuccess) {
        e = vr_launch_gather_sub(v->d_bv, nb, v->d_sub, v->last_mode, d_pix, npix, d_out, 0);
        v->launches++;
    }
    if (e == cudaSuccess) e = cudaDeviceSynchronize();
    if (e == cudaSuccess) e = cudaMemcpy(sub_out, d_out, sizeof(float) * 4 * (size_t)npix * nb, cudaMemcpyDeviceToHost);
    cudaFree(d_pix);
    cudaFree(d_out);
    VR_CUDA(v, e);
    return VR_OK;
}

extern "C" int vr_debug_stats(vr_volume* v, vr_stats* out) {
    if (!v) return fail(NULL, VR_ERR_INVALID_ARG, "vr_debug_stats: NULL handle");
    if (!out) return fail(v, VR_ERR_INVALID_ARG, "vr_debug_stats: NULL output");
    if (!v->last_stats_valid) return fail(v, VR_ERR_STATE, "vr_debug_stats: no vr_render since the last debug call");
    VR_CUDA(v, cudaDeviceSynchronize());
    VrViewState vs;
    VR_CUDA(v, cudaMemcpy(&vs, v->d_vs, sizeof(vs), cudaMemcpyDeviceToHost));
    out->samples = v->counting ? (int64_t)vs.samples : -1;
    out->rays = (int64_t)vs.total_sub_pixels;
    out->work_items = vs.total_items;
    out->subimage_bytes = (int64_t)vs.total_sub_pixels * (v->last_mode == VR_ALPHA ? 16 : 4);
    out->cells_touched = out->sectors_touched = out->lines_touched = -1;
    if (v->counting == 2) {
        unsigned long long c2[3] = {0, 0, 0};
        VR_CUDA(v, cudaMemset(v->d_counts2, 0, sizeof(c2)));
        VR_CUDA(v, vr_launch_count_bits(v->d_bitmap, v->bitmap_words, v->d_counts2, 0));
        v->launches++;
        VR_CUDA(v, cudaMemcpy(c2, v->d_counts2, sizeof(c2), cudaMemcpyDeviceToHost));
        out->cells_touched = (int64_t)c2[0];
        out->sectors_touched = (int64_t)c2[1];
        out->lines_touched = (int64_t)c2[2];
    }
    out->nbricks = v->grid.nbricks;
    out->overflow = vs.overflow;
    out->bricks_culled = vs.culled;
    out->ms_setup = out->ms_raycast = out->ms_composite = -1.0f;
    if (v->timing && v->timed_frames > 0) {
        cudaEvent_t* ev = v->ev[(v->timed_frames - 1) % VR_EV_RING];
        VR_CUDA(v, cudaEventElapsedTime(&out->ms_setup, ev[0], ev[1]));
        VR_CUDA(v, cudaEventElapsedTime(&out->ms_raycast, ev[1], ev[2]));
        VR_CUDA(v, cudaEventElapsedTime(&out->ms_composite, ev[2], ev[3]));
    }
    return VR_OK;
}

extern "C" int vr_debug_stage_times(vr_volume* v, int nframes, float* ms_out) {
    if (!v) return fail(NULL, VR_ERR_INVALID_ARG, "vr_debug_stage_times: NULL handle");
    if (!ms_out || nframes <= 0 || nframes > VR_EV_RING)
        return fail(v, VR_ERR_INVALID_ARG, "vr_debug_stage_times: need 1 <= nframes <= %d and an output", VR_EV_RING);
    if (!v->timing || v->timed_frames < nframes)
        return fail(v, VR_ERR_STATE, "vr_debug_stage_times: only %lld frames rendered since vr_set_timing(1)", v->timed_frames);
    VR_CUDA(v, cudaDeviceSynchronize());
    for (int f = 0; f < nframes; ++f) {
        cudaEvent_t* ev = v->ev[(v->timed_frames - nframes + f) % VR_EV_RING];
        for (int s3 = 0; s3 < 3; ++s3) VR_CUDA(v, cudaEventElapsedTime(ms_out + 3 * f + s3, ev[s3], ev[s3 + 1]));
    }
    return VR_OK;
}
