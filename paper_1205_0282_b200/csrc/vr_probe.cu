/*
 * vr_probe.cu -- DRAM fetch-granularity probe (debug export vr_debug_probe_dram; DESIGN.md
 * "What the hardware fetches"). Not on the frame path: it measures the machine property that
 * bounds the ray-cast kernel on sparsely sampled cubes (c3: rays ~6 voxels apart, every
 * 2x2x2 fetch misses L2), namely what ONE missed 4-byte load costs in DRAM bytes and how many
 * such misses per second the memory system sustains.
 *
 * Every thread issues `loads_per_thread` independent 4-byte loads (addresses come from a
 * counter-based hash, never from loaded data, 8 in flight per thread) at 32-byte-aligned
 * offsets of a caller-supplied buffer far larger than L2. Loads come in GROUPS: the loads of
 * one group fall into the same aligned `span`-byte block, in `group` DISTINCT 128-byte lines
 * of it (group = 1, span = 128: every load a random line; group = 2, span = 256: both halves
 * of a 256-byte pair; larger spans test DRAM-page locality). The load flavour is a template
 * parameter (cache operators and the L2 prefetch-size hints of PTX).
 * DRAM bytes per load = dram__bytes_read.sum of the launch (ncu) / loads; rate = loads / time.
 */
#include <stdio.h>
#include <string.h>

#include "vr_internal.cuh"

enum {
    PF_LD = 0,        /* ld.global.f32 (default .ca) */
    PF_NC,            /* ld.global.nc.f32: what __ldg emits, the ray-cast kernel's load */
    PF_CG,            /* ld.global.cg */
    PF_CS,            /* ld.global.cs */
    PF_CV,            /* ld.global.cv */
    PF_NC_NOALLOC,    /* ld.global.nc.L1::no_allocate */
    PF_NC_L2_64,      /* ld.global.nc.L1::no_allocate.L2::64B */
    PF_NC_L2_128,     /* ld.global.nc.L2::128B */
    PF_NC_L2_256,     /* ld.global.nc.L2::256B */
    PF_NC_V4,         /* ld.global.nc.v4.f32: 16 bytes per load */
    PF_NC_L2_64_ONLY, /* ld.global.nc.L2::64B (L1 allocates) */
    PF_TEX_F32,       /* tex1Dfetch<float> through a texture object over the (linear) buffer: the texture unit's path */
    PF_TEX_V4,        /* tex1Dfetch<float4>: 16 bytes per fetch */
    PF_ARR_V4_POINT,  /* tex3D<float4>, point sampling, from a 3-D CUDA array (block-linear; the probe allocates it, buf is not read) */
    PF_ARR_F32_LINEAR,/* tex3D<float>, linear filter, random position in a 3-D CUDA array: the texture arm's fetch */
    PF_COUNT
};

template <int F>
__device__ __forceinline__ float probe_load(const float* p, const float* base, cudaTextureObject_t tex) {
    float v, v1, v2, v3;
    if (F == PF_TEX_F32) return tex1Dfetch<float>(tex, (int)(p - base));
    if (F == PF_TEX_V4) {
        const float4 q = tex1Dfetch<float4>(tex, (int)((p - base) >> 2));
        return q.x + q.y + q.z + q.w;
    }
    if (F == PF_LD) asm volatile("ld.global.f32 %0, [%1];" : "=f"(v) : "l"(p));
    else if (F == PF_NC) asm volatile("ld.global.nc.f32 %0, [%1];" : "=f"(v) : "l"(p));
    else if (F == PF_CG) asm volatile("ld.global.cg.f32 %0, [%1];" : "=f"(v) : "l"(p));
    else if (F == PF_CS) asm volatile("ld.global.cs.f32 %0, [%1];" : "=f"(v) : "l"(p));
    else if (F == PF_CV) asm volatile("ld.global.cv.f32 %0, [%1];" : "=f"(v) : "l"(p));
    else if (F == PF_NC_NOALLOC) asm volatile("ld.global.nc.L1::no_allocate.f32 %0, [%1];" : "=f"(v) : "l"(p));
    else if (F == PF_NC_L2_64) asm volatile("ld.global.nc.L1::no_allocate.L2::64B.f32 %0, [%1];" : "=f"(v) : "l"(p));
    else if (F == PF_NC_L2_128) asm volatile("ld.global.nc.L2::128B.f32 %0, [%1];" : "=f"(v) : "l"(p));
    else if (F == PF_NC_L2_256) asm volatile("ld.global.nc.L2::256B.f32 %0, [%1];" : "=f"(v) : "l"(p));
    else if (F == PF_NC_L2_64_ONLY) asm volatile("ld.global.nc.L2::64B.f32 %0, [%1];" : "=f"(v) : "l"(p));
    else {
        asm volatile("ld.global.nc.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v), "=f"(v1), "=f"(v2), "=f"(v3) : "l"(p));
        v += v1 + v2 + v3;
    }
    return v;
}

__device__ __forceinline__ unsigned long long probe_mix(unsigned long long x) {
    x ^= x >> 33;
    x *= 0xff51afd7ed558ccdull;
    x ^= x >> 33;
    x *= 0xc4ceb9fe1a85ec53ull;
    x ^= x >> 33;
    return x;
}

/* nblocks = span-byte blocks of the buffer; lines = 128-byte lines per block (span / 128, >= 1);
 * group <= lines. Load i of a thread: group number i / group picks the block, i % group the line
 * (a hashed start line plus i % group, modulo lines: distinct within the group), a hashed
 * 32-byte sector inside the line (16-byte loads: sector-aligned too). */
template <int F>
__global__ void __launch_bounds__(256) vr_probe_dram_kernel(const float* __restrict__ buf, unsigned long long nblocks, int lines,
                                                            int span_floats, int group, int loads_per_thread, unsigned seed,
                                                            float* __restrict__ sink, cudaTextureObject_t tex) {
    const unsigned long long tid = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x;
    float acc = 0.0f;
    for (int i0 = 0; i0 < loads_per_thread; i0 += 8) {
        const float* p[8];
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            const int i = i0 + u;
            const unsigned long long h = probe_mix((tid << 24) ^ (unsigned long long)(i / group) ^ ((unsigned long long)seed << 48));
            const unsigned long long blk = h % nblocks;
            const unsigned line = (unsigned)(((h >> 40) + (unsigned)(i % group)) % (unsigned)lines);
            const unsigned sector = (unsigned)(probe_mix(h + (unsigned)(i % group) + 1u) & 3u);
            p[u] = buf + blk * (unsigned long long)span_floats + line * 32u + sector * 8u;
        }
#pragma unroll
        for (int u = 0; u < 8; ++u) acc += probe_load<F>(p[u], buf, tex);
    }
    if (acc == 1.2345e-30f) sink[0] = acc; /* keeps the loads alive; never true for the zero / finite data used */
}

/* 3-D array flavours: every fetch at a hashed texel (point sampling: its centre; linear filter: anywhere in its cell) */
template <int F>
__global__ void __launch_bounds__(256) vr_probe_array_kernel(cudaTextureObject_t tex, int ex, int ey, int ez, int loads_per_thread,
                                                             unsigned seed, float* __restrict__ sink) {
    const unsigned long long tid = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x;
    float acc = 0.0f;
    for (int i0 = 0; i0 < loads_per_thread; i0 += 8) {
        float x[8], y[8], z[8];
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            const unsigned long long h = probe_mix((tid << 24) ^ (unsigned long long)(i0 + u) ^ ((unsigned long long)seed << 48));
            const float f = F == PF_ARR_F32_LINEAR ? (float)((h >> 56) & 255u) * (1.0f / 256.0f) : 0.5f;
            x[u] = (float)(unsigned)(h % (unsigned)ex) + f;
            y[u] = (float)(unsigned)((h >> 20) % (unsigned)ey) + f;
            z[u] = (float)(unsigned)((h >> 40) % (unsigned)ez) + f;
        }
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            if (F == PF_ARR_V4_POINT) {
                const float4 q = tex3D<float4>(tex, x[u], y[u], z[u]);
                acc += q.x + q.y + q.z + q.w;
            } else {
                acc += tex3D<float>(tex, x[u], y[u], z[u]);
            }
        }
    }
    if (acc == 1.2345e-30f) sink[0] = acc;
}

typedef void (*probe_fn)(const float*, unsigned long long, int, int, int, int, unsigned, float*, cudaTextureObject_t);

extern "C" int vr_debug_probe_dram(const void* buf, uint64_t bytes, int flavour, int span_bytes, int group, int loads_per_thread,
                                   int ctas, int l2_fetch_granularity, float* ms_out, uint64_t* loads_out, void* stream) {
    if (!ms_out || !loads_out) return VR_ERR_INVALID_ARG;
    if (!buf && flavour != PF_ARR_V4_POINT && flavour != PF_ARR_F32_LINEAR) return VR_ERR_INVALID_ARG;
    if (flavour < 0 || flavour >= PF_COUNT) return VR_ERR_INVALID_ARG;
    if (span_bytes < 128 || (span_bytes & (span_bytes - 1)) || group < 1 || group > span_bytes / 128) return VR_ERR_INVALID_ARG;
    if (loads_per_thread < 8 || (loads_per_thread % 8) || (loads_per_thread % group) || ctas < 1) return VR_ERR_INVALID_ARG;
    if (bytes < (uint64_t)span_bytes) return VR_ERR_INVALID_ARG;
    static const probe_fn table[PF_COUNT] = {
        vr_probe_dram_kernel<PF_LD>, vr_probe_dram_kernel<PF_NC>, vr_probe_dram_kernel<PF_CG>, vr_probe_dram_kernel<PF_CS>,
        vr_probe_dram_kernel<PF_CV>, vr_probe_dram_kernel<PF_NC_NOALLOC>, vr_probe_dram_kernel<PF_NC_L2_64>,
        vr_probe_dram_kernel<PF_NC_L2_128>, vr_probe_dram_kernel<PF_NC_L2_256>, vr_probe_dram_kernel<PF_NC_V4>,
        vr_probe_dram_kernel<PF_NC_L2_64_ONLY>, vr_probe_dram_kernel<PF_TEX_F32>, vr_probe_dram_kernel<PF_TEX_V4>, NULL, NULL};
    cudaStream_t st = (cudaStream_t)stream;
    if (l2_fetch_granularity == 32 || l2_fetch_granularity == 64 || l2_fetch_granularity == 128) {
        if (cudaDeviceSetLimit(cudaLimitMaxL2FetchGranularity, (size_t)l2_fetch_granularity) != cudaSuccess) {
            cudaGetLastError();
            return VR_ERR_CUDA;
        }
    } else if (l2_fetch_granularity != 0) {
        return VR_ERR_INVALID_ARG;
    }
    float* sink = NULL;
    cudaEvent_t e0 = NULL, e1 = NULL;
    cudaError_t e = cudaMalloc(&sink, sizeof(float));
    if (e == cudaSuccess) e = cudaEventCreate(&e0);
    if (e == cudaSuccess) e = cudaEventCreate(&e1);
    /* texture flavours: a texture object over the buffer's head, as far as a linear-memory texture reaches (a device limit
     * in ELEMENTS: float4 texels reach four times as far as float ones); the probed range shrinks to it */
    cudaTextureObject_t tex = 0;
    if (e == cudaSuccess && (flavour == PF_TEX_F32 || flavour == PF_TEX_V4)) {
        const size_t el = flavour == PF_TEX_V4 ? 16 : 4;
        int dev = 0, max_el = 0;
        e = cudaGetDevice(&dev);
        if (e == cudaSuccess) e = cudaDeviceGetAttribute(&max_el, cudaDevAttrMaxTexture1DLinearWidth, dev);
        if (e == cudaSuccess) {
            if (bytes > (uint64_t)max_el * el) bytes = (uint64_t)max_el * el;
            if (bytes > ((uint64_t)1 << 31) * el / 1) bytes = ((uint64_t)1 << 31) * el; /* int texel index */
            cudaResourceDesc res;
            memset(&res, 0, sizeof(res));
            res.resType = cudaResourceTypeLinear;
            res.res.linear.devPtr = const_cast<void*>(buf);
            res.res.linear.desc = flavour == PF_TEX_V4 ? cudaCreateChannelDesc<float4>() : cudaCreateChannelDesc<float>();
            res.res.linear.sizeInBytes = (size_t)bytes;
            cudaTextureDesc td;
            memset(&td, 0, sizeof(td));
            td.readMode = cudaReadModeElementType;
            e = cudaCreateTextureObject(&tex, &res, &td, NULL);
        }
    }
    cudaArray_t arr = NULL;
    int ex = 0, ey = 0, ez = 0;
    if (e == cudaSuccess && (flavour == PF_ARR_V4_POINT || flavour == PF_ARR_F32_LINEAR)) {
        const size_t el = flavour == PF_ARR_V4_POINT ? 16 : 4;
        ex = ey = 1024;
        uint64_t slices = bytes / (el * 1024 * 1024);
        ez = (int)(slices > 2048 ? 2048 : (slices < 1 ? 1 : slices));
        const cudaChannelFormatDesc fmt = flavour == PF_ARR_V4_POINT ? cudaCreateChannelDesc<float4>() : cudaCreateChannelDesc<float>();
        e = cudaMalloc3DArray(&arr, &fmt, make_cudaExtent((size_t)ex, (size_t)ey, (size_t)ez), 0);
        if (e == cudaSuccess) {
            cudaResourceDesc res;
            memset(&res, 0, sizeof(res));
            res.resType = cudaResourceTypeArray;
            res.res.array.array = arr;
            cudaTextureDesc td;
            memset(&td, 0, sizeof(td));
            td.addressMode[0] = td.addressMode[1] = td.addressMode[2] = cudaAddressModeClamp;
            td.filterMode = flavour == PF_ARR_F32_LINEAR ? cudaFilterModeLinear : cudaFilterModePoint;
            td.readMode = cudaReadModeElementType;
            e = cudaCreateTextureObject(&tex, &res, &td, NULL);
        }
    }
    const unsigned long long nblocks = bytes / (uint64_t)span_bytes;
    const int lines = span_bytes / 128;
    if (e == cudaSuccess && arr) {
        if (flavour == PF_ARR_V4_POINT) {
            vr_probe_array_kernel<PF_ARR_V4_POINT><<<ctas, 256, 0, st>>>(tex, ex, ey, ez, loads_per_thread, 1u, sink);
            e = cudaEventRecord(e0, st);
            vr_probe_array_kernel<PF_ARR_V4_POINT><<<ctas, 256, 0, st>>>(tex, ex, ey, ez, loads_per_thread, 2u, sink);
        } else {
            vr_probe_array_kernel<PF_ARR_F32_LINEAR><<<ctas, 256, 0, st>>>(tex, ex, ey, ez, loads_per_thread, 1u, sink);
            e = cudaEventRecord(e0, st);
            vr_probe_array_kernel<PF_ARR_F32_LINEAR><<<ctas, 256, 0, st>>>(tex, ex, ey, ez, loads_per_thread, 2u, sink);
        }
        if (e == cudaSuccess) e = cudaEventRecord(e1, st);
        if (e == cudaSuccess) e = cudaGetLastError();
        if (e == cudaSuccess) e = cudaEventSynchronize(e1);
        if (e == cudaSuccess) e = cudaEventElapsedTime(ms_out, e0, e1);
    } else if (e == cudaSuccess) { /* one untimed launch (different addresses), then the timed one */
        table[flavour]<<<ctas, 256, 0, st>>>((const float*)buf, nblocks, lines, span_bytes / 4, group, loads_per_thread, 1u, sink, tex);
        e = cudaEventRecord(e0, st);
        table[flavour]<<<ctas, 256, 0, st>>>((const float*)buf, nblocks, lines, span_bytes / 4, group, loads_per_thread, 2u, sink, tex);
        if (e == cudaSuccess) e = cudaEventRecord(e1, st);
        if (e == cudaSuccess) e = cudaGetLastError();
        if (e == cudaSuccess) e = cudaEventSynchronize(e1);
        if (e == cudaSuccess) e = cudaEventElapsedTime(ms_out, e0, e1);
    }
    *loads_out = (uint64_t)ctas * 256ull * (uint64_t)loads_per_thread;
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    if (tex) cudaDestroyTextureObject(tex);
    if (arr) cudaFreeArray(arr);
    cudaFree(sink);
    if (e != cudaSuccess) {
        cudaGetLastError();
        return VR_ERR_CUDA;
    }
    return VR_OK;
}
