/*
 * vr_fused.cu -- fused front-to-back traversal: one ray per
 * frame pixel walks the bricks it crosses in order, with ONE accumulator, and writes the frame
 * directly. No sub-images, no compositing pass, and early ray termination is GLOBAL: a ray
 * that is opaque after its first brick never touches the bricks behind it.
 *
 * PAPER.md:152 (sec. 2.3.2) is the march of one ray through "the bounding cube" until the exit
 * point, the maximum or the opacity is reached; the paper splits that march into sub-cubes
 * only because its cube does not fit one GPU (:105, :113) and then pays for sub-frames and
 * compositing (:114, :156-184). On one B200 the whole cube is resident, so the split is only a
 * memory layout: the sample schedule is the ray's own (R5: anchored at the entry into the
 * whole volume), each sample is read from the brick that owns it (R6; ghosts make it
 * seam-free, R3), and the result is what the sort-last path gives for a single brick covering
 * the volume (R17) - with early termination ON as well, which sort-last cannot offer (R8).
 *
 * Work decomposition: persistent warps pull 8x4-pixel tiles of the FRAME (one atomic per
 * tile). Per ray: FP64 set-up once; per brick crossed: the owner brick of the next sample and
 * the integer sample range it owns (the same exact arithmetic as vr_raycast.cu), then the
 * float32 lattice march of vr_march.cuh.
 */
#include "vr_march.cuh"

#ifndef VR_TEX_DEPTH
#define VR_TEX_DEPTH 4 /* texture fetches a lane keeps in flight (as in vr_raycast.cu) */
#endif

template <int MODE, int LAY, bool CLAMP, bool COUNT, bool SKIP, bool TEX>
__global__ void __launch_bounds__(VR_RAYCAST_THREADS, VR_MIN_CTAS)
vr_fused_kernel(const VrRaycastParams prm, float4* __restrict__ frame) {
    extern __shared__ float4 s_lut[]; /* (entry, delta) pairs: shading (ALPHA), final colour map (MIP) */
    __shared__ double s_minv[16];

    const VrGrid& g = prm.grid;
    const int lane = threadIdx.x & 31;
    for (int i = threadIdx.x; i < prm.lut.n; i += blockDim.x) {
        s_lut[2 * i] = prm.lut.base[i];
        s_lut[2 * i + 1] = prm.lut.delta[i];
    }
    if (threadIdx.x < 16) s_minv[threadIdx.x] = prm.vs->Minv[threadIdx.x];
    __syncthreads();
    if (prm.vs->singular) return;

    const int W = prm.vs->W, H = prm.vs->H;
    /* tiles are handed out block by block (4 x 8 tiles = 32 x 32 pixels, row-major inside a block) so that
     * the warps in flight work on neighbouring rays - the same bricks and lines - instead of one frame row */
    const int tiles_x = (W + VR_TILE_W - 1) / VR_TILE_W, tiles_y = (H + VR_TILE_H - 1) / VR_TILE_H;
    const int blocks_x = (tiles_x + 3) >> 2, blocks_y = (tiles_y + 7) >> 3;
    const unsigned total = (unsigned)(blocks_x * blocks_y) << 5;
    const double step = prm.step;
    const float tau = prm.tau;
    LutView lut;
    lut.base = (unsigned)__cvta_generic_to_shared(s_lut);
    asm volatile("" : "+r"(lut.base));
    const float mip_stop = fminf(prm.lut.vmax, prm.vs->data_max);
    unsigned long long nsamples = 0;

    unsigned next = 0;
    if (lane == 0) next = atomicAdd(&prm.vs_rw->work_counter, 1u);
    next = __shfl_sync(FULL_MASK, next, 0);

    while (next < total) {
        const int item = (int)next;
        if (lane == 0) next = atomicAdd(&prm.vs_rw->work_counter, 1u);
        const int blk = item >> 5, by = blk / blocks_x, bx = blk - by * blocks_x;
        const int tx = (bx << 2) + (item & 3), ty = (by << 3) + ((item >> 2) & 7);
        const int pi = tx * VR_TILE_W + (lane & 7), pj = ty * VR_TILE_H + (lane >> 3);
        const bool in_frame = pi < W && pj < H; /* also false for the tiles a ragged block has beyond the frame */

        RaySetup ray;
        ray.K = 0;
        ray.step = step;
        if (in_frame) ray_setup(s_minv, W, H, pi, pj, g, step, ray);
        float stepf = (float)ray.step; /* path length a lattice sample stands for */
        asm volatile("" : "+f"(stepf)); /* one register: not re-converted from the double in every loop trip */

        Accum acc;
        acc.r = (MODE == VR_MIP) ? -INFINITY : 0.0f;
        acc.g = acc.b = acc.a = 0.0f;
        int stopped = (MODE == VR_ALPHA) ? !(acc.a < tau) : 0; /* int, not bool: no byte packing in the loop control */
        int k = 0; /* next sample of the ray's schedule */

        /* one trip per brick the ray crosses */
        while (__any_sync(FULL_MASK, k < ray.K && !stopped)) {
            const bool live = k < ray.K && !stopped;
            int bc[3] = {0, 0, 0}, blo[3], bhi[3], ext[3];
            int k_lo = k, k_hi = k + 1;
            bool owned = false;
            if (live) {
                double s, w;
                owned = sample_sw(ray, k, s, w); /* an empty interval is dropped (R5) */
                if (owned) {
#pragma unroll
                    for (int a = 0; a < 3; ++a) bc[a] = owner_axis(ray, g, s, a); /* R6: the brick that owns sample k */
                }
            }
            vr_brick_core(g, bc, blo, bhi);
#pragma unroll
            for (int a = 0; a < 3; ++a) ext[a] = bhi[a] - blo[a] + 2 * g.ghost;
            if (owned) {
                brick_range(ray, g, bc, blo, bhi, k_lo, k_hi);
                if (k_hi <= k) k_hi = k + 1; /* cannot happen (sample k is owned by bc); guarantees progress */
            }
            const int b = (bc[2] * g.g[1] + bc[1]) * g.g[0] + bc[0];
            const int slot_b = vr_slot_of_coords(g, bc); /* = b unless the handle is a part (row f3) */
            const float* __restrict__ brick = prm.bricks + (long long)slot_b * g.slot;
            asm volatile("" : "+l"(brick)); /* keep the base in registers: do not rebuild it per load */

            /* a brick the set-up kernel found transparent (R16: empty rendering rectangle) contributes exact
             * zeros: its samples are skipped, the schedule moves on to the next brick */
            if (owned && prm.bv[b].rx1 <= prm.bv[b].rx0) owned = false;
            const int k_lat = min(k_hi, max(k, ray.K - 2));
            int n = owned ? k_lat - k : 0;
            Lattice L;
            long long D[3];
            if (n > 0) {
                double s, w;
                sample_sw(ray, k, s, w);
#pragma unroll
                for (int a = 0; a < 3; ++a) {
                    const double p = VR_FMA(s, ray.d[a], ray.o[a]);
                    L.q[a] = to_fixed(p - ((double)(blo[a] - g.ghost) + 0.5));
                    D[a] = to_fixed(ray.step * ray.d[a]);
                }
            } else {
                L.q[0] = L.q[1] = L.q[2] = 0;
                D[0] = D[1] = D[2] = 0;
            }
            int active = n > 0 && !stopped;
            /* texture arm (vr_set_sampler; vr_raycast.cu has the reasoning): the lanes whose brick holds no blanked voxel
             * fetch through the brick's texture object - PER LANE here, the rays of a warp may be in different bricks
             * (the hardware serves the distinct objects of a warp one after the other) - VR_TEX_DEPTH fetches in flight;
             * the others fall through to the hand-rolled loop below */
            bool use_tex = false;
            cudaTextureObject_t tex = 0;
            if (TEX && MODE == VR_ALPHA) {
                use_tex = owned && __ldg(prm.tex_nan + slot_b) == 0;
                tex = use_tex ? __ldg(prm.tex + slot_b) : 0;
                const double h = 1.0 / 4294967296.0;
                float P0x = (float)((double)L.q[0] * h + 0.5), P0y = (float)((double)L.q[1] * h + 0.5), P0z = (float)((double)L.q[2] * h + 0.5);
                float Dfx = (float)((double)D[0] * h), Dfy = (float)((double)D[1] * h), Dfz = (float)((double)D[2] * h);
                asm volatile("" : "+f"(P0x), "+f"(P0y), "+f"(P0z), "+f"(Dfx), "+f"(Dfy), "+f"(Dfz));
                const int n0 = n;
                int tactive = active && use_tex;
                const unsigned* __restrict__ tbits = SKIP ? prm.cell_bits + (long long)slot_b * prm.cell_words : NULL;
                int tpm = -1;
                bool ttransp = false;
                while (__any_sync(FULL_MASK, tactive)) {
                    if (tactive) {
                        if (SKIP) { /* macro-cell look-ups need the lattice: one sample per trip */
                            const int cx = (int)(L.q[0] >> 32), cy = (int)(L.q[1] >> 32), cz = (int)(L.q[2] >> 32);
                            const int m = ((cz >> 3) * prm.nc[1] + (cy >> 3)) * prm.nc[0] + (cx >> 3);
                            if (m != tpm) {
                                tpm = m;
                                ttransp = (__ldg(tbits + (m >> 5)) >> (m & 31)) & 1u;
                            }
                            int adv = 1;
                            if (ttransp) {
                                adv = leap_steps(L, D, n);
                            } else {
                                const float kf = (float)(n0 - n);
                                float v = tex3D<float>(tex, fmaf(kf, Dfx, P0x), fmaf(kf, Dfy, P0y), fmaf(kf, Dfz, P0z));
                                float4 c = classify_alpha(v, lut, prm.lut);
                                if (c.w > prm.tex_guard) { /* R20's guard (vr_raycast.cu): nearly opaque entries at steps < 1 */
                                    v = trilinear<LAY, 0, CLAMP, false>(brick, g, ext, L, prm.bitmap, (long long)slot_b * g.slot);
                                    c = classify_alpha(v, lut, prm.lut);
                                }
                                if (COUNT) nsamples += (v == v) ? 1 : 0;
                                blend_alpha(acc, v, stepf, c);
                                stopped = !(acc.a < tau);
                            }
                            L.q[0] += D[0] * adv, L.q[1] += D[1] * adv, L.q[2] += D[2] * adv;
                            n -= adv;
                            tactive = n > 0 && !stopped;
                        } else {
                            const float kf = (float)(n0 - n);
                            float vq[VR_TEX_DEPTH];
#pragma unroll
                            for (int u = 0; u < VR_TEX_DEPTH; ++u) {
                                const float ku = kf + (float)u;
                                vq[u] = tex3D<float>(tex, fmaf(ku, Dfx, P0x), fmaf(ku, Dfy, P0y), fmaf(ku, Dfz, P0z));
                            }
                            bool by_hand = false;
#pragma unroll
                            for (int u = 0; u < VR_TEX_DEPTH; ++u) {
                                if (tactive && !by_hand) {
                                    const float4 c = classify_alpha(vq[u], lut, prm.lut);
                                    if (c.w > prm.tex_guard) {
                                        by_hand = true; /* R20's guard (vr_raycast.cu): the rest of the batch is dropped and fetched again */
                                    } else {
                                        if (COUNT) nsamples += (vq[u] == vq[u]) ? 1 : 0;
                                        blend_alpha(acc, vq[u], stepf, c);
                                        stopped = !(acc.a < tau);
                                        --n;
                                        tactive = n > 0 && !stopped;
                                    }
                                }
                            }
                            if (by_hand) { /* this loop does not advance the lattice */
                                Lattice Lj;
                                const long long jj = (long long)(n0 - n);
                                Lj.q[0] = L.q[0] + D[0] * jj, Lj.q[1] = L.q[1] + D[1] * jj, Lj.q[2] = L.q[2] + D[2] * jj;
                                const float v = trilinear<LAY, 0, CLAMP, false>(brick, g, ext, Lj, prm.bitmap, (long long)slot_b * g.slot);
                                if (COUNT) nsamples += (v == v) ? 1 : 0;
                                shade_alpha(acc, v, stepf, lut, prm.lut);
                                stopped = !(acc.a < tau);
                                --n;
                                tactive = n > 0 && !stopped;
                            }
                        }
                    }
                }
                if (use_tex) active = 0; /* done (n == 0 or stopped); the other lanes still have their samples to take */
            }
            Corners C;
            int pcx = INT_MIN, pcy = 0, pcz = 0;
            /* R19: samples based in a transparent macro-cell are skipped (see vr_raycast.cu) */
            const unsigned* __restrict__ cbits = (SKIP && MODE == VR_ALPHA) ? prm.cell_bits + (long long)slot_b * prm.cell_words : NULL;
            const float2* __restrict__ cmm = (SKIP && MODE == VR_MIP) ? prm.cell_mm + (long long)slot_b * (prm.nc[0] * prm.nc[1] * prm.nc[2]) : NULL;
            float pbound = INFINITY;
            int pm = -1;
            bool ptransp = false;
            while (__any_sync(FULL_MASK, active)) {
                if (active) {
                    const int cx = (int)(L.q[0] >> 32), cy = (int)(L.q[1] >> 32), cz = (int)(L.q[2] >> 32);
                    int adv = 1; /* lattice steps this trip takes */
                    if (!VR_REUSE || cx != pcx || cy != pcy || cz != pcz) {
                        if (SKIP) {
                            const int m = ((cz >> 3) * prm.nc[1] + (cy >> 3)) * prm.nc[0] + (cx >> 3);
                            if (MODE == VR_ALPHA) {
                                if (m != pm) {
                                    pm = m;
                                    ptransp = (__ldg(cbits + (m >> 5)) >> (m & 31)) & 1u;
                                }
                            } else {
                                /* MIP: no sample based in this macro-cell can exceed its maximum (plus a rounding margin of the
                                 * float32 interpolation); if that cannot raise the ray's maximum, the cell is stepped over */
                                if (m != pm) {
                                    pm = m;
                                    const float cmax = __ldg(&cmm[m].y);
                                    pbound = cmax + fabsf(cmax) * 1e-6f;
                                }
                                ptransp = pbound <= acc.r;
                            }
                            if (ptransp) adv = -leap_steps(L, D, n); /* negative: a leap over samples that cannot matter, nothing fetched */
                        }
                        if (adv > 0) {
                            fetch8<LAY, 0, CLAMP, COUNT>(brick, g, ext, L, prm.bitmap, (long long)slot_b * g.slot, C);
                            pcx = cx, pcy = cy, pcz = cz;
                        }
                    }
                    if (adv > 0) {
                        float v = lerp8(C, L);
                        if (v != v) v = lerp8_blanked(C, L); /* R14: some of the 8 voxels are blanked (rare path) */
                        if (COUNT) nsamples += (v == v) ? 1 : 0; /* R14: a dropped sample is NaN */
                        if (MODE == VR_MIP) {
                            acc.r = fmaxf(acc.r, v);
                            stopped = acc.r >= mip_stop;
                        } else {
                            shade_alpha(acc, v, stepf, lut, prm.lut);
                            stopped = !(acc.a < tau);
                        }
                        L.q[0] += D[0], L.q[1] += D[1], L.q[2] += D[2];
                    } else {
                        adv = -adv;
                        L.q[0] += D[0] * adv, L.q[1] += D[1] * adv, L.q[2] += D[2] * adv;
                    }
                    n -= adv;
                    active = n > 0 && !stopped;
                }
            }
            /* the (at most two) samples next to the exit point, one by one in FP64 (R5) */
            if (live) {
                for (int kk = max(k_lat, k); owned && kk < k_hi && !stopped; ++kk) {
                    double s, w;
                    if (!sample_sw(ray, kk, s, w)) continue;
#pragma unroll
                    for (int a = 0; a < 3; ++a) {
                        const double p = VR_FMA(s, ray.d[a], ray.o[a]);
                        L.q[a] = to_fixed(p - ((double)(blo[a] - g.ghost) + 0.5));
                    }
                    float v;
                    if (TEX && use_tex && prm.tex_only) { /* a released store has no float32 cells: the exit samples through the array too */
                        const double h = 1.0 / 4294967296.0;
                        v = tex3D<float>(tex, (float)((double)L.q[0] * h + 0.5), (float)((double)L.q[1] * h + 0.5), (float)((double)L.q[2] * h + 0.5));
                    } else {
                        v = trilinear<LAY, 0, CLAMP, COUNT>(brick, g, ext, L, prm.bitmap, (long long)slot_b * g.slot);
                    }
                    if (COUNT) nsamples += (v == v) ? 1 : 0;
                    if (MODE == VR_MIP) {
                        acc.r = fmaxf(acc.r, v);
                        stopped = acc.r >= mip_stop;
                    } else {
                        shade_alpha(acc, v, (float)w, lut, prm.lut);
                        stopped = !(acc.a < tau);
                    }
                }
                k = k_hi;
            }
        }

        if (in_frame) {
            float4 o;
            if (MODE == VR_ALPHA) {
                o = make_float4(acc.r, acc.g, acc.b, acc.a);
            } else if (acc.r == -INFINITY) {
                o = make_float4(0.0f, 0.0f, 0.0f, 0.0f); /* R11: the ray took no sample */
            } else {
                const float u = __saturatef((acc.r - prm.lut.vmin) * prm.lut.inv_range);
                const float x = u * prm.lut.scale;
                const int i = min((int)x, prm.lut.nm2);
                const float f = x - (float)i;
                const float4 e = s_lut[2 * i], d = s_lut[2 * i + 1];
                o = make_float4(fmaf(f, d.x, e.x), fmaf(f, d.y, e.y), fmaf(f, d.z, e.z), 1.0f);
            }
            __stcs(frame + ((long long)pj * W + pi), o);
        }
        next = __shfl_sync(FULL_MASK, next, 0);
    }
    if (COUNT) {
        for (int o = 16; o > 0; o >>= 1) nsamples += __shfl_xor_sync(FULL_MASK, nsamples, o);
        if (lane == 0 && nsamples) atomicAdd(&prm.vs_rw->samples, nsamples);
    }
}

template <int MODE, int LAY, bool CLAMP, bool COUNT, bool SKIP = false, bool TEX = false>
static cudaError_t launch_fused(const VrRaycastParams& p, float* frame, long long items, cudaStream_t st) {
    const size_t smem = 2 * sizeof(float4) * (size_t)p.lut.n;
    /* asked of the runtime at every launch (a few microseconds): no process-wide cache to go stale across devices or threads */
    int dev = 0, sms = 0, cached_per_sm = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (e == cudaSuccess)
        e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&cached_per_sm, vr_fused_kernel<MODE, LAY, CLAMP, COUNT, SKIP, TEX>,
                                                          VR_RAYCAST_THREADS, smem);
    if (e != cudaSuccess) return e;
    if (cached_per_sm < 1) return cudaErrorLaunchOutOfResources;
    long long ctas = (long long)sms * cached_per_sm;
    const long long want = (items + (VR_RAYCAST_THREADS / 32) - 1) / (VR_RAYCAST_THREADS / 32);
    if (ctas > want) ctas = want < 1 ? 1 : want;
    vr_fused_kernel<MODE, LAY, CLAMP, COUNT, SKIP, TEX><<<(int)ctas, VR_RAYCAST_THREADS, smem, st>>>(p, reinterpret_cast<float4*>(frame));
    return cudaGetLastError();
}

template <int MODE, bool COUNT>
static cudaError_t launch_fused_mode(const VrRaycastParams& p, float* frame, long long items, cudaStream_t st) {
    const bool clamp = p.grid.ghost == 0;
    const VrGrid& g = p.grid;
    const bool t442 = g.layout == VR_LAYOUT_TILED && g.tl[0] == 2 && g.tl[1] == 2 && g.tl[2] == 1 && g.ml[0] == 0 && g.ml[1] == 0 &&
                      g.ml[2] == 0;
    if (g.layout == VR_LAYOUT_LINEAR)
        return clamp ? launch_fused<MODE, LAY_LINEAR, true, COUNT>(p, frame, items, st)
                     : launch_fused<MODE, LAY_LINEAR, false, COUNT>(p, frame, items, st);
    if (t442 && MODE == VR_ALPHA && p.tex != NULL && p.bitmap == NULL) { /* texture arm (vr_set_sampler): VR_ALPHA only */
        if (!clamp && p.cell_bits != NULL) return launch_fused<VR_ALPHA, LAY_TILE442, false, COUNT, true, true>(p, frame, items, st);
        return clamp ? launch_fused<VR_ALPHA, LAY_TILE442, true, COUNT, false, true>(p, frame, items, st)
                     : launch_fused<VR_ALPHA, LAY_TILE442, false, COUNT, false, true>(p, frame, items, st);
    }
    if (t442) {
        if (!clamp && (MODE == VR_ALPHA ? p.cell_bits != NULL : p.cell_mm != NULL)) /* R19: macro-cell skipping */
            return launch_fused<MODE, LAY_TILE442, false, COUNT, true>(p, frame, items, st);
        return clamp ? launch_fused<MODE, LAY_TILE442, true, COUNT>(p, frame, items, st)
                     : launch_fused<MODE, LAY_TILE442, false, COUNT>(p, frame, items, st);
    }
    return clamp ? launch_fused<MODE, LAY_GENERIC, true, COUNT>(p, frame, items, st)
                 : launch_fused<MODE, LAY_GENERIC, false, COUNT>(p, frame, items, st);
}

cudaError_t vr_launch_fused(const VrRaycastParams& p, float* frame, int W, int H, bool count, cudaStream_t st) {
    const long long tiles_x = (W + VR_TILE_W - 1) / VR_TILE_W, tiles_y = (H + VR_TILE_H - 1) / VR_TILE_H;
    const long long items = ((tiles_x + 3) / 4) * ((tiles_y + 7) / 8) * 32;
    if (p.mode == VR_ALPHA)
        return count ? launch_fused_mode<VR_ALPHA, true>(p, frame, items, st) : launch_fused_mode<VR_ALPHA, false>(p, frame, items, st);
    return count ? launch_fused_mode<VR_MIP, true>(p, frame, items, st) : launch_fused_mode<VR_MIP, false>(p, frame, items, st);
}
