/*
 * vr_debug.cu -- test exports: per-ray brick lists (R10) and sub-image read-back (row a8).
 *
 * Ray-brick list of a pixel (each ray is intersected with the sub-cube's
 * bounding cube; "a few rays may pass the rendering rectangle test but still do not
 * intersect"): the bricks whose core box [lo,hi) (closed on the volume's outer high faces,
 * R4) overlaps the ray's clipped segment [t0,t1] with positive length, by increasing entry
 * distance, ties by brick index. All of it is IEEE double arithmetic with individually
 * rounded operations (vr_view.cuh), in the order DESIGN.md "Set-up arithmetic" fixes.
 */
#include "vr_view.cuh"

struct DbgRay {
    double o[3], d[3];
    double tfar;
};

/* R1, R2: same operations, in the same order, as the ray-cast kernel's ray set-up. */
__device__ void dbg_pixel_ray(const double* Minv, int W, int H, int i, int j, DbgRay& r) {
    const double x = VR_SUB(VR_DIV(VR_MUL(2.0, VR_ADD((double)i, 0.5)), (double)W), 1.0);
    const double y = VR_SUB(VR_DIV(VR_MUL(2.0, VR_ADD((double)j, 0.5)), (double)H), 1.0);
    double nr[4], fr[4];
    for (int k = 0; k < 4; ++k) {
        const double xy = VR_ADD(VR_MUL(Minv[k], x), VR_MUL(Minv[4 + k], y));
        const double w = VR_MUL(Minv[12 + k], 1.0);
        nr[k] = VR_ADD(VR_ADD(xy, VR_MUL(Minv[8 + k], -1.0)), w);
        fr[k] = VR_ADD(VR_ADD(xy, VR_MUL(Minv[8 + k], 1.0)), w);
    }
    double len = 0.0;
    for (int a = 0; a < 3; ++a) {
        const double na = VR_DIV(nr[a], nr[3]);
        const double fa = VR_DIV(fr[a], fr[3]);
        r.o[a] = na;
        r.d[a] = VR_SUB(fa, na);
        len = VR_ADD(len, VR_MUL(r.d[a], r.d[a]));
    }
    len = VR_SQRT(len);
    for (int a = 0; a < 3; ++a) r.d[a] = VR_DIV(r.d[a], len);
    r.tfar = len;
}

/* R4 slab test against [lo,hi) (closed where closed_hi[a]); margin = smallest decision margin. */
__device__ bool dbg_slab(const DbgRay& r, const double lo[3], const double hi[3], const bool closed_hi[3], double& tin,
                         double& tout, double& margin) {
    double t0 = -INFINITY, t1 = INFINITY, mg = INFINITY;
    for (int a = 0; a < 3; ++a) {
        if (r.d[a] == 0.0) {
            const bool inside = (r.o[a] >= lo[a]) && (closed_hi[a] ? (r.o[a] <= hi[a]) : (r.o[a] < hi[a]));
            const double m = fmin(fabs(VR_SUB(r.o[a], lo[a])), fabs(VR_SUB(r.o[a], hi[a])));
            if (m < mg) mg = m;
            if (!inside) {
                margin = mg;
                return false;
            }
        } else {
            double ta = VR_DIV(VR_SUB(lo[a], r.o[a]), r.d[a]);
            double tb = VR_DIV(VR_SUB(hi[a], r.o[a]), r.d[a]);
            if (ta > tb) {
                const double t = ta;
                ta = tb;
                tb = t;
            }
            if (ta > t0) t0 = ta;
            if (tb < t1) t1 = tb;
        }
    }
    tin = t0;
    tout = t1;
    const double m = fabs(VR_SUB(t1, t0));
    if (m < mg) mg = m;
    margin = mg;
    return t1 >= t0;
}

__global__ void vr_ray_bricks_kernel(VrGrid g, const VrViewState* __restrict__ vs, const int* __restrict__ pixels, int npix,
                                     int* __restrict__ counts, int* __restrict__ lists, double* __restrict__ tins, int maxlen,
                                     unsigned char* __restrict__ grazing) {
    const int q = blockIdx.x * blockDim.x + threadIdx.x;
    if (q >= npix) return;
    DbgRay r;
    dbg_pixel_ray(vs->Minv, vs->W, vs->H, pixels[2 * q], pixels[2 * q + 1], r);
    const double glo[3] = {0.0, 0.0, 0.0}, ghi[3] = {(double)g.n[0], (double)g.n[1], (double)g.n[2]};
    const bool gclosed[3] = {true, true, true};
    double tin, tout, mg;
    bool gz = false;
    int cnt = 0;
    const bool hit = dbg_slab(r, glo, ghi, gclosed, tin, tout, mg);
    if (mg < 1e-9) gz = true;
    const double t0 = tin > 0.0 ? tin : 0.0, t1 = tout < r.tfar ? tout : r.tfar;
    int* lst = lists + (long long)q * maxlen;
    double* tl = tins + (long long)q * maxlen;
    for (int x = 0; x < maxlen; ++x) lst[x] = -1;
    if (hit && t1 > t0) {
        for (int b = 0; b < g.nbricks; ++b) {
            int bc[3], lo[3], hi[3];
            vr_brick_coords(g, b, bc);
            vr_brick_core(g, bc, lo, hi);
            double blo[3], bhi[3];
            bool bcl[3];
            for (int a = 0; a < 3; ++a) {
                blo[a] = (double)lo[a];
                bhi[a] = (double)hi[a];
                bcl[a] = hi[a] == g.n[a];
            }
            double bi, bo, bm;
            const bool bh = dbg_slab(r, blo, bhi, bcl, bi, bo, bm);
            if (!bh) {
                if (bm < 1e-9) gz = true;
                continue;
            }
            const double a0 = bi > t0 ? bi : t0, a1 = bo < t1 ? bo : t1;
            if (fabs(VR_SUB(a1, a0)) < 1e-9) gz = true;
            if (a1 > a0) {
                /* stable insertion by entry distance (bricks arrive in ascending index) */
                if (cnt < maxlen) {
                    int y = cnt - 1;
                    while (y >= 0 && tl[y] > a0) {
                        tl[y + 1] = tl[y];
                        lst[y + 1] = lst[y];
                        --y;
                    }
                    tl[y + 1] = a0;
                    lst[y + 1] = b;
                }
                ++cnt;
            }
        }
        const int m = cnt < maxlen ? cnt : maxlen;
        for (int x = 1; x < m; ++x)
            if (fabs(VR_SUB(tl[x], tl[x - 1])) < 1e-9) gz = true;
    }
    counts[q] = cnt;
    if (grazing) grazing[q] = gz ? 1 : 0;
}

cudaError_t vr_launch_ray_bricks(const VrGrid& grid, const VrViewState* vs, const int* d_pixels, int npix, int* d_counts,
                                 int* d_lists, double* d_tins, int maxlen, unsigned char* d_grazing, cudaStream_t st) {
    vr_ray_bricks_kernel<<<(npix + 127) / 128, 128, 0, st>>>(grid, vs, d_pixels, npix, d_counts, d_lists, d_tins, maxlen,
                                                            d_grazing);
    return cudaGetLastError();
}

/* out[(q*nbricks + b)*4 ..]: the sub-image value brick b holds for listed pixel q. */
__global__ void vr_gather_sub_kernel(const VrBrickView* __restrict__ bv, int nbricks, const void* __restrict__ sub, int mode,
                                     const int* __restrict__ pixels, int npix, float4* __restrict__ out) {
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= (long long)npix * nbricks) return;
    const int q = (int)(t / nbricks), b = (int)(t % nbricks);
    const int i = pixels[2 * q], j = pixels[2 * q + 1];
    const VrBrickView v = bv[b];
    float4 o = (mode == VR_ALPHA) ? make_float4(0.f, 0.f, 0.f, 0.f) : make_float4(-INFINITY, 0.f, 0.f, 0.f);
    if (i >= v.rx0 && i < v.rx1 && j >= v.ry0 && j < v.ry1) {
        const long long off = v.sub_offset + (long long)(j - v.ly0) * (v.lx1 - v.lx0) + (i - v.lx0);
        if (mode == VR_ALPHA) o = reinterpret_cast<const float4*>(sub)[off];
        else o.x = reinterpret_cast<const float*>(sub)[off];
    }
    out[t] = o;
}

cudaError_t vr_launch_gather_sub(const VrBrickView* bv, int nbricks, const void* sub, int mode, const int* d_pixels, int npix,
                                 float* d_out, cudaStream_t st) {
    const long long n = (long long)npix * nbricks;
    vr_gather_sub_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(bv, nbricks, sub, mode, d_pixels, npix,
                                                                     reinterpret_cast<float4*>(d_out));
    return cudaGetLastError();
}

/* Test export: the padded cells of brick b as a dense [dz][dy][dx] box (any layout). */
__global__ void vr_brick_copy_kernel(VrGrid g, const float* __restrict__ bricks, int b, int dx, int dy, int dz,
                                     float* __restrict__ out) {
    const long long n = (long long)dx * dy * dz;
    const float* __restrict__ src = bricks + (long long)vr_slot_index(g, b) * g.slot;
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < n; t += (long long)gridDim.x * blockDim.x) {
        const int i = (int)(t % dx), j = (int)((t / dx) % dy), k = (int)(t / ((long long)dx * dy));
        out[t] = src[vr_cell_offset(g, i, j, k)];
    }
}

cudaError_t vr_launch_brick_copy(const VrGrid& grid, const float* bricks, int b, const int dims[3], float* d_out,
                                 cudaStream_t st) {
    vr_brick_copy_kernel<<<148 * 8, 256, 0, st>>>(grid, bricks, b, dims[0], dims[1], dims[2], d_out);
    return cudaGetLastError();
}

/* Touched-cells bitmap (bench instrumentation): out3[0] += set bits (distinct brick-store
 * cells read), out3[1] += non-zero bytes (distinct 32-byte sectors: 8 consecutive cells),
 * out3[2] += non-zero words (distinct 128-byte lines: 32 consecutive cells). */
__global__ void vr_count_bits_kernel(const unsigned* __restrict__ bitmap, long long words, unsigned long long* __restrict__ out3) {
    unsigned long long cells = 0, sectors = 0, lines = 0;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < words; i += (long long)gridDim.x * blockDim.x) {
        const unsigned w = bitmap[i];
        cells += __popc(w);
        sectors += ((w & 0xffu) != 0) + ((w & 0xff00u) != 0) + ((w & 0xff0000u) != 0) + ((w & 0xff000000u) != 0);
        lines += (w != 0);
    }
    for (int o = 16; o > 0; o >>= 1) {
        cells += __shfl_xor_sync(0xffffffffu, cells, o);
        sectors += __shfl_xor_sync(0xffffffffu, sectors, o);
        lines += __shfl_xor_sync(0xffffffffu, lines, o);
    }
    if ((threadIdx.x & 31) == 0) {
        atomicAdd(out3, cells);
        atomicAdd(out3 + 1, sectors);
        atomicAdd(out3 + 2, lines);
    }
}

cudaError_t vr_launch_count_bits(const unsigned* bitmap, long long words, unsigned long long* d_out3, cudaStream_t st) {
    vr_count_bits_kernel<<<148 * 8, 256, 0, st>>>(bitmap, words, d_out3);
    return cudaGetLastError();
}
