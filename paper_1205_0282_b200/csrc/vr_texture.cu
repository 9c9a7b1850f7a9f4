/*
 * vr_texture.cu -- the texture-object arm of the brick store.
 *
 * PAPER.md:150 (sec. 2.3.2): the sub-cube is kept in the GPU's texture memory so that the
 * built-in tri-linear interpolation can be used; :69 names the same facility. north_star asks
 * for the bricks "either as 3D CUDA arrays behind texture objects or as a tiled linear layout with
 * hand-rolled vectorised trilinear interpolation, whichever ncu shows is faster": this is the
 * first arm.
 *
 * One 3-D CUDA array per brick of the handle, extent = the brick's ghost-padded extent, float32
 * texels, behind a texture object with linear filtering, clamp addressing and unnormalised
 * coordinates: texel i is centred at i + 1/2 and the hardware interpolates between the two nearest
 * centres - R3's convention exactly, with the padded cell index as the texel index. The arrays
 * are a second copy of the brick store, filled from it on the device through surface objects
 * (vr_tex_fill_kernel) after an upload; the hand-rolled path keeps the float32 store, which
 * VR_MIP needs for its values (the hardware filter's 8 fractional weight bits cannot meet MIP's 1e-5: MIP frames use
 * the arrays only to rule out the samples that cannot be a ray's maximum, vr_raycast.cu), and which
 * VR_ALPHA keeps using for bricks that hold blanked (NaN) voxels: the filter cannot apply R14's rule.
 */
#include <cuda_fp16.h>
#include <string.h>

#include <new>

#include "vr_view.cuh"

struct VrTexStore {
    int n;                      /* bricks of the handle (slots) */
    cudaArray_t* arr;
    cudaTextureObject_t* tex;
    cudaSurfaceObject_t* surf;
    cudaTextureObject_t* d_tex; /* device copies of the two tables */
    cudaSurfaceObject_t* d_surf;
    int3* d_ext;                /* padded extent of every slot */
    int* d_nan;                 /* 1 where the slot holds a NaN (blanked) voxel: such bricks are sampled by hand (R14) */
    int texel;                  /* VR_TEXEL_FLOAT, or - the exact MIP filter only - VR_TEXEL_HALF / VR_TEXEL_BYTE */
};

void vr_tex_destroy(VrTexStore* t) {
    if (!t) return;
    for (int s = 0; s < t->n; ++s) {
        if (t->tex && t->tex[s]) cudaDestroyTextureObject(t->tex[s]);
        if (t->surf && t->surf[s]) cudaDestroySurfaceObject(t->surf[s]);
        if (t->arr && t->arr[s]) cudaFreeArray(t->arr[s]);
    }
    cudaFree(t->d_tex);
    cudaFree(t->d_surf);
    cudaFree(t->d_ext);
    cudaFree(t->d_nan);
    delete[] t->arr;
    delete[] t->tex;
    delete[] t->surf;
    delete t;
    cudaGetLastError();
}

/* brick held in slot s of the handle's store (the inverse of vr_slot_index) */
static __host__ __device__ int brick_of_slot(const VrGrid& g, int s) {
    if (!g.part) return s;
    const int w = g.pb1[0] - g.pb0[0], h = g.pb1[1] - g.pb0[1];
    const int bx = g.pb0[0] + s % w, by = g.pb0[1] + (s / w) % h, bz = g.pb0[2] + s / (w * h);
    return (bz * g.g[1] + by) * g.g[0] + bx;
}

/* the store's host tables and device tables, no array yet */
static cudaError_t tex_alloc(const VrGrid& g, VrTexStore** out, int texel) {
    *out = NULL;
    VrTexStore* t = new (std::nothrow) VrTexStore();
    if (!t) return cudaErrorMemoryAllocation;
    memset(t, 0, sizeof(*t));
    t->n = g.nown;
    t->texel = texel;
    t->arr = new (std::nothrow) cudaArray_t[g.nown]();
    t->tex = new (std::nothrow) cudaTextureObject_t[g.nown]();
    t->surf = new (std::nothrow) cudaSurfaceObject_t[g.nown]();
    cudaError_t e = (t->arr && t->tex && t->surf) ? cudaSuccess : cudaErrorMemoryAllocation;
    if (e == cudaSuccess) e = cudaMalloc(&t->d_tex, sizeof(cudaTextureObject_t) * g.nown);
    if (e == cudaSuccess) e = cudaMalloc(&t->d_surf, sizeof(cudaSurfaceObject_t) * g.nown);
    if (e == cudaSuccess) e = cudaMalloc(&t->d_ext, sizeof(int3) * g.nown);
    if (e == cudaSuccess) e = cudaMalloc(&t->d_nan, sizeof(int) * g.nown);
    if (e == cudaSuccess) e = cudaMemset(t->d_nan, 0, sizeof(int) * g.nown);
    if (e != cudaSuccess) {
        cudaGetLastError();
        vr_tex_destroy(t);
        return e;
    }
    *out = t;
    return cudaSuccess;
}

/* array, texture object and surface object of slot s; their handles and the slot's extent go to the device tables */
static cudaError_t tex_create_slot(VrTexStore* t, const VrGrid& g, int s) {
    int bc[3], lo[3], hi[3];
    vr_brick_coords(g, brick_of_slot(g, s), bc);
    vr_brick_core(g, bc, lo, hi);
    const int3 ext = make_int3(hi[0] - lo[0] + 2 * g.ghost, hi[1] - lo[1] + 2 * g.ghost, hi[2] - lo[2] + 2 * g.ghost);
    const cudaChannelFormatDesc fmt = t->texel == VR_TEXEL_HALF ? cudaCreateChannelDescHalf()
                                      : t->texel == VR_TEXEL_BYTE ? cudaCreateChannelDesc<unsigned char>() : cudaCreateChannelDesc<float>();
    cudaError_t e = cudaMalloc3DArray(&t->arr[s], &fmt, make_cudaExtent((size_t)ext.x, (size_t)ext.y, (size_t)ext.z), cudaArraySurfaceLoadStore);
    if (e != cudaSuccess) return e;
    cudaResourceDesc res;
    memset(&res, 0, sizeof(res));
    res.resType = cudaResourceTypeArray;
    res.res.array.array = t->arr[s];
    cudaTextureDesc td;
    memset(&td, 0, sizeof(td));
    td.addressMode[0] = td.addressMode[1] = td.addressMode[2] = cudaAddressModeClamp;
    td.filterMode = cudaFilterModeLinear;
    td.readMode = t->texel == VR_TEXEL_BYTE ? cudaReadModeNormalizedFloat : cudaReadModeElementType; /* byte q reads as q / 255 */
    td.normalizedCoords = 0;
    e = cudaCreateTextureObject(&t->tex[s], &res, &td, NULL);
    if (e == cudaSuccess) e = cudaCreateSurfaceObject(&t->surf[s], &res);
    if (e == cudaSuccess) e = cudaMemcpy(t->d_tex + s, t->tex + s, sizeof(cudaTextureObject_t), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(t->d_surf + s, t->surf + s, sizeof(cudaSurfaceObject_t), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(t->d_ext + s, &ext, sizeof(int3), cudaMemcpyHostToDevice);
    return e;
}

/* all = true: every slot's array at once (the second copy beside the store); false: tables only, the arrays come slot by
 * slot (vr_tex_convert_slot: vr_volume_release_store) */
cudaError_t vr_tex_create(const VrGrid& g, VrTexStore** out, bool all, int texel) {
    VrTexStore* t = NULL;
    cudaError_t e = tex_alloc(g, &t, texel);
    for (int s = 0; all && s < g.nown && e == cudaSuccess; ++s) e = tex_create_slot(t, g, s);
    if (e != cudaSuccess) {
        cudaGetLastError();
        vr_tex_destroy(t);
        *out = NULL;
        return e;
    }
    *out = t;
    return cudaSuccess;
}

const cudaTextureObject_t* vr_tex_table(const VrTexStore* t) { return t ? t->d_tex : NULL; }
const int* vr_tex_nan_table(const VrTexStore* t) { return t ? t->d_nan : NULL; }
int vr_tex_texel(const VrTexStore* t) { return t ? t->texel : VR_TEXEL_FLOAT; }

/* Padded cell (i, j, k) of slot s -> texel (i, j, k) of the slot's array. A CTA takes the 4 x 2 rows
 * (j, k) of one row of micro-tiles, one row per warp, lanes along x, so the eight warps together consume
 * whole 128-byte lines of the store (L1 serves a line's other rows to the neighbouring warps); the surface
 * write is coalesced. Once per upload. */
template <int TEXEL>
__global__ void __launch_bounds__(256)
vr_tex_fill_kernel(VrGrid g, const float* __restrict__ bricks, const cudaSurfaceObject_t* __restrict__ surf,
                   const int3* __restrict__ ext, int* __restrict__ has_nan, int slot0, const float2* __restrict__ brick_mm) {
    const int s = blockIdx.y + slot0;
    /* byte texels: q = round(255 (v - min) / (max - min)) with the brick's range (row f1's table); a constant brick gets q = 0 */
    float q_lo = 0.0f, q_scale = 0.0f;
    if (TEXEL == VR_TEXEL_BYTE) {
        const float2 mm = brick_mm[brick_of_slot(g, s)];
        q_lo = mm.x;
        q_scale = mm.y > mm.x ? 255.0f / (mm.y - mm.x) : 0.0f;
    }
    const int3 e = ext[s];
    const cudaSurfaceObject_t su = surf[s];
    const float* __restrict__ src = bricks + (long long)s * g.slot;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int nj = (e.y + 3) >> 2, nk = (e.z + 1) >> 1;
    bool nan_seen = false;
    for (int blk = blockIdx.x; blk < nj * nk; blk += gridDim.x) {
        const int j = ((blk % nj) << 2) + (warp & 3), k = ((blk / nj) << 1) + (warp >> 2);
        if (j >= e.y || k >= e.z) continue;
        const unsigned row = vr_axis_offset(g.ax[1], j) + vr_axis_offset(g.ax[2], k);
        for (int i = lane; i < e.x; i += 32) {
            const float v = __ldcs(src + row + vr_axis_offset(g.ax[0], i));
            nan_seen = nan_seen || v != v;
            if (TEXEL == VR_TEXEL_HALF) surf3Dwrite(__half_as_ushort(__float2half_rn(v)), su, i * 2, j, k); /* to nearest: |h - v| <= 2^-11 |v| + 2^-25 */
            else if (TEXEL == VR_TEXEL_BYTE) surf3Dwrite((unsigned char)__float2uint_rn(fminf(fmaxf((v - q_lo) * q_scale, 0.0f), 255.0f)), su, i, j, k);
            else surf3Dwrite(v, su, i * 4, j, k);
        }
    }
    /* R14: the hardware filter cannot apply the blanking rule (it drops a NaN corner whose 8-bit weight rounds to
     * zero, the rule drops the SAMPLE from a weight of 4e-6 on): bricks with blanked voxels keep the hand-rolled sampler */
    if (__any_sync(0xffffffffu, nan_seen) && lane == 0) has_nan[s] = 1;
}

static cudaError_t launch_fill(const VrGrid& grid, const float* bricks, const VrTexStore* t, int slot0, int nslots, const float2* brick_mm,
                               cudaStream_t st) {
    const int nj = (grid.P + 3) >> 2, nk = (grid.P + 1) >> 1;
    long long bx = (long long)nj * nk;
    if (bx > 4096) bx = 4096;
    cudaError_t e = cudaMemsetAsync(t->d_nan + slot0, 0, sizeof(int) * nslots, st);
    if (e != cudaSuccess) return e;
    const dim3 gr((unsigned)bx, (unsigned)nslots);
    if (t->texel == VR_TEXEL_BYTE && !brick_mm) return cudaErrorInvalidValue;
    if (t->texel == VR_TEXEL_HALF) vr_tex_fill_kernel<VR_TEXEL_HALF><<<gr, 256, 0, st>>>(grid, bricks, t->d_surf, t->d_ext, t->d_nan, slot0, brick_mm);
    else if (t->texel == VR_TEXEL_BYTE) vr_tex_fill_kernel<VR_TEXEL_BYTE><<<gr, 256, 0, st>>>(grid, bricks, t->d_surf, t->d_ext, t->d_nan, slot0, brick_mm);
    else vr_tex_fill_kernel<VR_TEXEL_FLOAT><<<gr, 256, 0, st>>>(grid, bricks, t->d_surf, t->d_ext, t->d_nan, slot0, brick_mm);
    return cudaGetLastError();
}

cudaError_t vr_launch_tex_fill(const VrGrid& grid, const float* bricks, const VrTexStore* t, const float2* brick_mm, cudaStream_t st) {
    return launch_fill(grid, bricks, t, 0, t->n, brick_mm, st);
}

/* vr_volume_release_store, one slot: create the slot's array, fill it from the store, wait, and say whether the slot holds
 * blanked voxels (then its float32 cells must stay: R14 needs them). */
cudaError_t vr_tex_convert_slot(const VrGrid& grid, const float* bricks, VrTexStore* t, int s, int* has_nan, cudaStream_t st) {
    cudaError_t e = tex_create_slot(t, grid, s);
    if (e == cudaSuccess) e = launch_fill(grid, bricks, t, s, 1, NULL, st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(has_nan, t->d_nan + s, sizeof(int), cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    return e;
}

/* R23's constant, measured: the largest |filtered fetch - exact tri-linear value| over n hashed positions inside slot s,
 * the exact value in double from the float32 store. Positions are texel coordinates in [1/2, extent - 1/2): inside the
 * volume of texel centres, as every sample of a frame is. dec_a / dec_b decode an 8-bit fetch ((max - min), min; else 1, 0). */
__global__ void __launch_bounds__(256)
vr_tex_error_kernel(VrGrid g, const float* __restrict__ bricks, const cudaTextureObject_t* __restrict__ tex, const int3* __restrict__ ext,
                    int s, long long n, unsigned seed, float dec_a, float dec_b, float* __restrict__ max_err) {
    const int3 e = ext[s];
    const cudaTextureObject_t t = tex[s];
    const float* __restrict__ src = bricks + (long long)s * g.slot;
    float worst = 0.0f;
    for (long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x; q < n; q += (long long)gridDim.x * blockDim.x) {
        unsigned long long h = ((unsigned long long)seed << 40) ^ (unsigned long long)q;
        float p[3];
        const int ee[3] = {e.x, e.y, e.z};
        for (int a = 0; a < 3; ++a) {
            h ^= h >> 33; h *= 0xff51afd7ed558ccdull; h ^= h >> 33; h *= 0xc4ceb9fe1a85ec53ull; h ^= h >> 33;
            p[a] = 0.5f + (float)((double)(h >> 11) * (1.0 / 9007199254740992.0) * (double)(ee[a] - 1));
            if (p[a] >= (float)ee[a] - 0.5f) p[a] = (float)ee[a] - 0.5f - 1e-3f;
        }
        const float f = fmaf(tex3D<float>(t, p[0], p[1], p[2]), dec_a, dec_b);
        int c[3];
        double w[3];
        for (int a = 0; a < 3; ++a) {
            const double u = (double)p[a] - 0.5;
            c[a] = (int)floor(u);
            if (c[a] > ee[a] - 2) c[a] = ee[a] - 2;
            w[a] = u - (double)c[a];
        }
        double v[2][2][2];
        for (int k = 0; k < 2; ++k)
            for (int j = 0; j < 2; ++j)
                for (int i = 0; i < 2; ++i)
                    v[k][j][i] = (double)src[vr_axis_offset(g.ax[0], c[0] + i) + vr_axis_offset(g.ax[1], c[1] + j) + vr_axis_offset(g.ax[2], c[2] + k)];
        double x[2][2];
        for (int k = 0; k < 2; ++k)
            for (int j = 0; j < 2; ++j) x[k][j] = v[k][j][0] + w[0] * (v[k][j][1] - v[k][j][0]);
        const double y0 = x[0][0] + w[1] * (x[0][1] - x[0][0]), y1 = x[1][0] + w[1] * (x[1][1] - x[1][0]);
        const double exact = y0 + w[2] * (y1 - y0);
        const float err = (float)fabs((double)f - exact);
        if (err == err) worst = fmaxf(worst, err);
    }
    for (int o = 16; o > 0; o >>= 1) worst = fmaxf(worst, __shfl_xor_sync(0xffffffffu, worst, o));
    if ((threadIdx.x & 31) == 0) atomicMax(reinterpret_cast<int*>(max_err), __float_as_int(worst)); /* non-negative floats order as ints */
}

cudaError_t vr_launch_tex_error(const VrGrid& grid, const float* bricks, const VrTexStore* t, int s, long long n, unsigned seed, float dec_a,
                                float dec_b, float* max_err, cudaStream_t st) {
    vr_tex_error_kernel<<<148 * 4, 256, 0, st>>>(grid, bricks, t->d_tex, t->d_ext, s, n, seed, dec_a, dec_b, max_err);
    return cudaGetLastError();
}
