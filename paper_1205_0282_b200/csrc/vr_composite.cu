/*
 * vr_composite.cu -- sort-last compositing of sub-images into the final frame (SURVEY.md
 * sec. 8(a) row a9) and, for MIP, the final colour mapping.
 *
 * PAPER.md:170-174 (sec. 2.3.3): sub-frames are merged guided by their rendering rectangles;
 * the alpha blending operator is associative, so sub-images composite in visibility order;
 * MIP composites in any order; :172 the merged scalar frame is colour-mapped at the end.
 * :114 names compositing as the bottleneck of distributed image-order rendering, which is
 * why it is a bandwidth-shaped kernel here: every sub-image pixel is read once with
 * coalesced 16-byte loads and the frame is written once.
 *
 * One CTA per 32x8-pixel tile of the frame. The CTA first filters the layer table, in
 * visibility order, down to the layers whose rectangle meets its tile (ballot + prefix,
 * order-preserving), then each thread walks that short list for its pixel:
 *   ALPHA  C += (1-A) C_l,  A += (1-A) A_l      (float32, R15; no early termination)
 *   MIP    m = max(m, m_l); at the end RGB = LUT(u(m)), A = 1, or (0,0,0,0) if m = -inf (R11)
 * Row f3 (multi-GPU sort-last): a part's MIP frame leaves as the raw maximum, ONE float per
 * pixel as in the paper (:180: 4 MB per 1024^2 sub-frame; VR_MIP_RAW: m, or -inf without a sample), and the
 * partial frames of the parts are merged by the same kernel (ALPHA: `over` in part order; VR_MIP_PARTS: maximum
 * of the scalar pieces, then the colour mapping). The output may be a WINDOW of the frame (a rectangle stored
 * [h][w]): a part composites its sub-images straight into the rectangle-packed pieces it sends (:184).
 */
#include "vr_internal.cuh"

#define COMP_THREADS (VR_COMP_TILE_W * VR_COMP_TILE_H)
#define COMP_LIST 256
#ifndef VR_COMP_UNROLL
#define VR_COMP_UNROLL 16 /* layers whose loads are in flight per pixel */
#endif
static constexpr int COMP_UNROLL = VR_COMP_UNROLL;

struct CompEntry {
    unsigned long long addr;
    int x0, y0, x1, y1;
    int sx0, sy0, pitch;
    int inside; /* the whole tile lies inside the layer's rectangle */
};

template <int MODE>
__global__ void __launch_bounds__(COMP_THREADS)
vr_composite_kernel(const VrCompLayer* __restrict__ layers, const int* __restrict__ order, int n, int4 win, VrLut lut,
                    void* __restrict__ out_, const int* __restrict__ bound) {
    /* win = (x0, y0, x1, y1): the pixels of the frame this launch writes, stored [y1-y0][x1-x0] at out_ */
    const int W = win.z, H = win.w, WP = win.z - win.x;
    __shared__ CompEntry s_list[COMP_LIST];
    __shared__ int s_warp_cnt[COMP_THREADS / 32];
    __shared__ int s_count;

    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const int tx0 = win.x + blockIdx.x * VR_COMP_TILE_W, ty0 = win.y + blockIdx.y * VR_COMP_TILE_H;
    float4* __restrict__ out = reinterpret_cast<float4*>(out_);
    const long long oidx = (long long)(ty0 + (int)(threadIdx.x / VR_COMP_TILE_W) - win.y) * WP + (tx0 + (int)(threadIdx.x & (VR_COMP_TILE_W - 1)) - win.x);
    const int tx1 = min(tx0 + VR_COMP_TILE_W, W), ty1 = min(ty0 + VR_COMP_TILE_H, H);
    const int px = tx0 + (tid & (VR_COMP_TILE_W - 1)), py = ty0 + tid / VR_COMP_TILE_W;
    const bool live = px < W && py < H;
    /* a tile outside the union of the layers' rectangles is blank: one load decides it, no table walk
     * (c3: the cube covers 18 % of a 1080p frame) */
    if (bound) {
        const int bx0 = __ldg(bound), by0 = __ldg(bound + 1), bx1 = __ldg(bound + 2), by1 = __ldg(bound + 3);
        if (!(bx0 < tx1 && bx1 > tx0 && by0 < ty1 && by1 > ty0)) {
            if (live) {
                if (MODE == VR_MIP_RAW) __stcs(reinterpret_cast<float*>(out_) + oidx, -INFINITY);
                else __stcs(out + oidx, make_float4(0.0f, 0.0f, 0.0f, 0.0f));
            }
            return;
        }
    }

    float cr = 0.0f, cg = 0.0f, cb = 0.0f, ca = 0.0f;
    float m = -INFINITY;

    for (int q0 = 0; q0 < n; q0 += COMP_THREADS) {
        /* order-preserving filter of up to 256 layers */
        const int q = q0 + tid;
        bool hit = false;
        VrCompLayer L;
        if (q < n) {
            L = layers[order[q]];
            hit = L.x0 < tx1 && L.x1 > tx0 && L.y0 < ty1 && L.y1 > ty0 && L.x1 > L.x0 && L.y1 > L.y0;
        }
        const unsigned bal = __ballot_sync(0xffffffffu, hit);
        if (lane == 0) s_warp_cnt[wid] = __popc(bal);
        __syncthreads();
        int base = 0;
        for (int w = 0; w < wid; ++w) base += s_warp_cnt[w];
        if (hit) {
            CompEntry e;
            e.addr = L.addr;
            e.x0 = L.x0; e.y0 = L.y0; e.x1 = L.x1; e.y1 = L.y1;
            e.sx0 = L.sx0; e.sy0 = L.sy0; e.pitch = L.pitch;
            e.inside = L.x0 <= tx0 && L.x1 >= tx1 && L.y0 <= ty0 && L.y1 >= ty1;
            s_list[base + __popc(bal & ((1u << lane) - 1u))] = e;
        }
        if (tid == COMP_THREADS - 1) s_count = base + __popc(bal);
        __syncthreads();
        const int cnt = s_count;

        if (live) {
#pragma unroll COMP_UNROLL
            for (int k = 0; k < cnt; ++k) {
                const CompEntry& e = s_list[k];
                const bool in = e.inside || (px >= e.x0 && px < e.x1 && py >= e.y0 && py < e.y1);
                if (in) {
                    const long long off = (long long)(py - e.sy0) * e.pitch + (px - e.sx0);
                    if (MODE == VR_ALPHA) {
                        const float4 s = __ldcs(reinterpret_cast<const float4*>(e.addr) + off);
                        const float t = 1.0f - ca;
                        cr = fmaf(t, s.x, cr);
                        cg = fmaf(t, s.y, cg);
                        cb = fmaf(t, s.z, cb);
                        ca = fmaf(t, s.w, ca);
                    } else { /* VR_MIP: brick sub-images; VR_MIP_RAW likewise; VR_MIP_PARTS: the parts' scalar pieces (-inf = no sample) */
                        m = fmaxf(m, __ldcs(reinterpret_cast<const float*>(e.addr) + off));
                    }
                }
            }
        }
        __syncthreads();
    }

    if (live && MODE == VR_MIP_RAW) {
        __stcs(reinterpret_cast<float*>(out_) + oidx, m);
    } else if (live) {
        float4 o;
        if (MODE == VR_ALPHA) {
            o = make_float4(cr, cg, cb, ca);
        } else if (m == -INFINITY) {
            o = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
        } else {
            const float u = __saturatef((m - lut.vmin) * lut.inv_range);
            const float x = u * (float)(lut.n - 1);
            const int i = min((int)x, lut.n - 2);
            const float f = x - (float)i;
            const float4 e = __ldg(lut.base + i), d = __ldg(lut.delta + i);
            o = make_float4(fmaf(f, d.x, e.x), fmaf(f, d.y, e.y), fmaf(f, d.z, e.z), 1.0f);
        }
        __stcs(out + oidx, o);
    }
}

cudaError_t vr_launch_composite(const VrCompLayer* layers, const int* order, int n, int W, int H, int mode,
                                const VrLut& lut, float* out, const int* bound, const int* window, cudaStream_t st) {
    const int4 win = window ? make_int4(window[0], window[1], window[2], window[3]) : make_int4(0, 0, W, H);
    if (win.z <= win.x || win.w <= win.y) return cudaSuccess; /* an empty window: nothing to write */
    dim3 grid((win.z - win.x + VR_COMP_TILE_W - 1) / VR_COMP_TILE_W, (win.w - win.y + VR_COMP_TILE_H - 1) / VR_COMP_TILE_H);
    if (mode == VR_ALPHA)
        vr_composite_kernel<VR_ALPHA><<<grid, COMP_THREADS, 0, st>>>(layers, order, n, win, lut, out, bound);
    else if (mode == VR_MIP)
        vr_composite_kernel<VR_MIP><<<grid, COMP_THREADS, 0, st>>>(layers, order, n, win, lut, out, bound);
    else if (mode == VR_MIP_RAW)
        vr_composite_kernel<VR_MIP_RAW><<<grid, COMP_THREADS, 0, st>>>(layers, order, n, win, lut, out, bound);
    else
        vr_composite_kernel<VR_MIP_PARTS><<<grid, COMP_THREADS, 0, st>>>(layers, order, n, win, lut, out, bound);
    return cudaGetLastError();
}

/* ------------------------------------------------------------------------------------------
 * vr_composite_static: stand-alone compositing (row a9) for callers that must not allocate - code under CUDA graph
 * capture, tight serving loops, harnesses that forbid cudaMalloc. vr_composite takes its two small device tables
 * (layer table, visibility order) from cudaMallocAsync; here they live in a file-scope __device__ array of a fixed,
 * modest size, which every GPU that loads the library holds until the process exits (11 KB). The kernel is the same.
 *
 * The array's name is a host-side stand-in in host code, not a device address: the address comes from
 * cudaGetSymbolAddress, once per device, with that device current.
 * Every call shares the array; it keeps the last call's tables. Nothing in it has to start at zero: a call rewrites
 * entries [0, n) of both tables and its kernel reads no others. Calls that overlap on the GPU (different streams, no
 * dependency between them) race on the tables; calls on one stream are ordered by it.
 */
#include <mutex>

#define VR_COMP_STATIC_MAX VR_COMPOSITE_STATIC_MAX_LAYERS
static __device__ __align__(256) unsigned char g_comp_scratch[VR_COMP_STATIC_MAX * sizeof(VrCompLayer) + VR_COMP_STATIC_MAX * sizeof(int)];

void vr_global_error(const char* fmt, ...); /* vr_api.cu: the message vr_last_error(NULL) returns */

#define COMP_MAX_DEVICES 64
static unsigned char* g_comp_scratch_addr[COMP_MAX_DEVICES]; /* device address of g_comp_scratch on each device, or NULL */
static std::mutex g_comp_scratch_lock;

/* device address of the scratch array on the CURRENT device (looked up on the first call per device) */
static cudaError_t comp_scratch_address(unsigned char** out) {
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= COMP_MAX_DEVICES) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> hold(g_comp_scratch_lock);
    if (!g_comp_scratch_addr[dev]) {
        void* p = NULL;
        e = cudaGetSymbolAddress(&p, g_comp_scratch);
        if (e != cudaSuccess) return e;
        g_comp_scratch_addr[dev] = static_cast<unsigned char*>(p);
    }
    *out = g_comp_scratch_addr[dev];
    return cudaSuccess;
}

extern "C" int vr_composite_static(const float* const* layers, const int* rects, const int* order, int n, int width, int height,
                                   float* out, void* stream) {
    if (!layers || !rects || !order || !out) {
        vr_global_error("vr_composite_static: NULL argument");
        return VR_ERR_INVALID_ARG;
    }
    if (n < 0 || n > VR_COMP_STATIC_MAX) {
        vr_global_error("vr_composite_static: n = %d layers, the static scratch holds at most %d (use vr_composite)", n, VR_COMP_STATIC_MAX);
        return VR_ERR_INVALID_ARG;
    }
    if (width <= 0 || height <= 0 || width > 32768 || height > 32768) {
        vr_global_error("vr_composite_static: bad frame size %dx%d", width, height);
        return VR_ERR_INVALID_ARG;
    }
    VrCompLayer tab[VR_COMP_STATIC_MAX]; /* host tables on the stack: no host allocation either */
    unsigned char seen[VR_COMP_STATIC_MAX];
    memset(seen, 0, sizeof(seen));
    for (int l = 0; l < n; ++l) {
        const int* r = rects + 4 * l;
        if (r[0] < 0 || r[1] < 0 || r[2] > width || r[3] > height || r[2] < r[0] || r[3] < r[1]) {
            vr_global_error("vr_composite_static: rectangle %d outside the viewport", l);
            return VR_ERR_INVALID_ARG;
        }
        if (!layers[l] && r[2] > r[0] && r[3] > r[1]) {
            vr_global_error("vr_composite_static: layer %d is NULL", l);
            return VR_ERR_INVALID_ARG;
        }
        if (order[l] < 0 || order[l] >= n || seen[order[l]]) {
            vr_global_error("vr_composite_static: order is not a permutation");
            return VR_ERR_INVALID_ARG;
        }
        seen[order[l]] = 1;
        VrCompLayer& L = tab[l];
        L.x0 = r[0]; L.y0 = r[1]; L.x1 = r[2]; L.y1 = r[3];
        L.sx0 = r[0]; L.sy0 = r[1];
        L.pitch = r[2] - r[0];
        L.pad = 0;
        L.addr = (unsigned long long)(uintptr_t)layers[l];
    }
    unsigned char* scratch = NULL;
    cudaError_t e = comp_scratch_address(&scratch);
    cudaStream_t st = (cudaStream_t)stream;
    VrCompLayer* d_tab = reinterpret_cast<VrCompLayer*>(scratch);
    int* d_order = reinterpret_cast<int*>(scratch + VR_COMP_STATIC_MAX * sizeof(VrCompLayer));
    /* pageable (stack) sources: the runtime has taken the bytes when the call returns; the writes are ordered on `st` */
    if (e == cudaSuccess && n > 0) e = cudaMemcpyAsync(d_tab, tab, sizeof(VrCompLayer) * n, cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess && n > 0) e = cudaMemcpyAsync(d_order, order, sizeof(int) * n, cudaMemcpyHostToDevice, st);
    VrLut none;
    memset(&none, 0, sizeof(none));
    if (e == cudaSuccess) e = vr_launch_composite(d_tab, d_order, n, width, height, VR_ALPHA, none, out, NULL, NULL, st);
    if (e != cudaSuccess) {
        cudaGetLastError();
        vr_global_error("vr_composite_static: %s", cudaGetErrorString(e));
        return VR_ERR_CUDA;
    }
    return VR_OK;
}
