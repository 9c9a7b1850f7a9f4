/*
 * vr_synth_cuda.cu -- device twin of the seeded input generator (see vr_synth.h).
 *
 * Needed because the largest workload (4096x4096x1536 float32, ~103 GB) cannot be
 * made on the host and pushed over PCIe in reasonable time. It uploads the tables the
 * CPU side built (vr_synth_cpu.c) and evaluates the very same vs_voxel() per element,
 * so the device cube is bit-identical to what the CPU oracle reads procedurally.
 * Input generation only: nothing of the renderer lives here.
 *
 * Build: nvcc -gencode arch=compute_100a,code=sm_100a -fmad=false (synth/build.py).
 */
#include <cuda_runtime.h>
#include <stdlib.h>
#include <string.h>
#include "vr_synth.h"

struct vs_dev_cube {
    vs_cube d;        /* struct with DEVICE pointers (passed to kernels by value) */
    void* blocks[13]; /* allocations to free */
    int nblocks;
};

template <typename T>
static const T* up(vs_dev_cube* h, const T* src, size_t n, cudaError_t* err) {
    if (n == 0) n = 1;
    void* p = nullptr;
    cudaError_t e = cudaMalloc(&p, n * sizeof(T));
    if (e != cudaSuccess) { *err = e; return nullptr; }
    h->blocks[h->nblocks++] = p;
    e = cudaMemcpy(p, src, n * sizeof(T), cudaMemcpyHostToDevice);
    if (e != cudaSuccess) *err = e;
    return (const T*)p;
}

extern "C" void vs_dev_cube_destroy(void* handle) {
    vs_dev_cube* h = (vs_dev_cube*)handle;
    if (!h) return;
    for (int i = 0; i < h->nblocks; ++i) cudaFree(h->blocks[i]);
    free(h);
}

extern "C" void* vs_dev_cube_create(const vs_cube* host, int64_t nprof, int64_t ncell, int64_t nitems) {
    vs_dev_cube* h = (vs_dev_cube*)calloc(1, sizeof(vs_dev_cube));
    h->d = *host;
    cudaError_t err = cudaSuccess;
    size_t ns = (size_t)host->nsrc;
    h->d.x0 = up(h, host->x0, ns, &err); h->d.y0 = up(h, host->y0, ns, &err); h->d.z0 = up(h, host->z0, ns, &err);
    h->d.lx = up(h, host->lx, ns, &err); h->d.ly = up(h, host->ly, ns, &err); h->d.lz = up(h, host->lz, ns, &err);
    h->d.ox = up(h, host->ox, ns, &err); h->d.oy = up(h, host->oy, ns, &err); h->d.oz = up(h, host->oz, ns, &err);
    h->d.peak = up(h, host->peak, ns, &err);
    h->d.prof = up(h, host->prof, (size_t)nprof, &err);
    h->d.cell_start = up(h, host->cell_start, (size_t)ncell + 1, &err);
    h->d.cell_items = up(h, host->cell_items, (size_t)nitems, &err);
    if (err != cudaSuccess) { vs_dev_cube_destroy(h); return nullptr; }
    return h;
}

__global__ void vs_fill_kernel(vs_cube c, float* __restrict__ dst, int64_t bx, int64_t by, int64_t bz,
                               int64_t sx, int64_t sy, int64_t sz) {
    int64_t n = sx * sy * sz;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        int64_t x = i % sx, t = i / sx;
        int64_t y = t % sy, z = t / sy;
        dst[i] = vs_voxel(&c, bx + x, by + y, bz + z);
    }
}

extern "C" int vs_dev_cube_fill(void* handle, float* d_dst, int64_t bx, int64_t by, int64_t bz,
                                int64_t sx, int64_t sy, int64_t sz, void* stream) {
    vs_dev_cube* h = (vs_dev_cube*)handle;
    if (!h || !d_dst || sx <= 0 || sy <= 0 || sz <= 0) return 1;
    int64_t n = sx * sy * sz;
    int64_t blocks = (n + 255) / 256;
    if (blocks > 148 * 64) blocks = 148 * 64;
    vs_fill_kernel<<<(unsigned)blocks, 256, 0, (cudaStream_t)stream>>>(h->d, d_dst, bx, by, bz, sx, sy, sz);
    return cudaGetLastError() == cudaSuccess ? 0 : 2;
}

__global__ void vs_layer_kernel(uint64_t seed, uint64_t layer, int64_t pix0, int64_t npix, float4* __restrict__ dst) {
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < npix; i += (int64_t)gridDim.x * blockDim.x) {
        float o[4];
        vs_layer_pixel(seed, layer, (uint64_t)(pix0 + i), o);
        dst[i] = make_float4(o[0], o[1], o[2], o[3]);
    }
}

extern "C" int vs_dev_layer_fill(uint64_t seed, int64_t layer, int64_t pix0, int64_t npix, float* d_dst, void* stream) {
    if (!d_dst || npix <= 0) return 1;
    int64_t blocks = (npix + 255) / 256;
    if (blocks > 148 * 32) blocks = 148 * 32;
    vs_layer_kernel<<<(unsigned)blocks, 256, 0, (cudaStream_t)stream>>>(seed, (uint64_t)layer, pix0, npix, (float4*)d_dst);
    return cudaGetLastError() == cudaSuccess ? 0 : 2;
}
