/*
 * vr_raycast.cu -- the per-brick ray-cast kernel.
 *
 * PAPER.md:152 (sec. 2.3.2): each GPU thread computes its ray's start and direction and its
 * intersection with the bounding cube, rays that miss leave at once, the ray is marched until
 * the exit point or until the opacity / the maximum value is reached; :69,:150 tri-linear
 * interpolation of the data; :45 transfer function -> colour and opacity accumulated along
 * the ray; :174 MIP. One thread = one pixel of one brick's rendering rectangle (:150).
 *
 * B200 design:
 *   - persistent grid (resident CTAs x 148 SMs); warps pull (brick, 8x4-pixel tile) work items
 *     from a device-built list with one atomic per item, bricks in visibility order so the
 *     tiles in flight share one or two bricks in L2;
 *   - ray, global clip and the integer sample range each brick owns are computed once per
 *     (ray, brick) in FP64 with individually rounded operations, so the kernel takes exactly
 *     the sample set the definition prescribes (R5, R6);
 *   - sample positions advance on a 32.32 fixed-point lattice in brick-local coordinates
 *     (two integer adds per axis and step): the integer word is the voxel index, the fraction
 *     word becomes the float32 interpolation weight with a shift/or - no FP64 and no
 *     int<->float conversion in the loop, and a position error below 1e-7 voxel;
 *   - tri-linear interpolation is hand-rolled in float32 on 8 read-only loads (hardware
 *     texture filtering has 8-bit weights and cannot meet the MIP tolerance);
 *   - the LUT is staged in dynamic shared memory as interleaved (entry, delta) pairs;
 *   - early ray termination and loop exit are warp votes;
 *   - 80 registers (3 CTAs per SM): the FP64 ray is rebuilt for the exit samples instead of
 *     living through the loop; the 8 voxels are kept while a ray stays in one cell;
 *   - with a transfer function that has a transparent range, samples based in a transparent
 *     8x8x8 macro-cell are not fetched (R19; the SKIP instances).
 * Measured bounds: DRAM lines on the 103 GB cube, issue slots / L1 data stage on the small
 * cubes (DESIGN.md sections 8 and 9; profiles/).
 */
#include "vr_march.cuh"

#ifndef VR_TEX_CTAS
#define VR_TEX_CTAS 3 /* resident CTAs per SM the texture-arm instances are cut for */
#endif
#ifndef VR_TEX_DEPTH
#define VR_TEX_DEPTH 4 /* texture fetches a lane keeps in flight */
#endif
#ifndef VR_MIP_TEX_DEPTH
#define VR_MIP_TEX_DEPTH 4 /* fetches a lane keeps in flight in the MIP filter loop */
#endif
#ifndef VR_MIP_QUEUE
#define VR_MIP_QUEUE 4 /* candidate samples a lane queues before the warp evaluates them by hand */
#endif
#ifndef VR_TEX_COPIES
#define VR_TEX_COPIES 8 /* copies of the table in the texture-arm instances (more CTAs per SM: less room for each) */
#endif

/* RAYTAB: every (ray, brick) segment starts from the frame's ray table (vr_rays.cu) - the dense views' choice: a quarter
 * of c2's instructions were the per-segment FP64 ray set-up. Sparse views (the 103 GB cube) are bound by DRAM requests,
 * not by issue slots: there the table's kernel (0.017 ms) costs more than it saves (0.002 ms), so their instances keep
 * the set-up inside (RAYTAB = false, prm.rays == NULL). The values are the same bit for bit either way. */
template <int MODE, int LAY, int PT, bool CLAMP, bool COUNT, bool SKIP, bool TEX, bool RAYTAB, bool GUARD>
__global__ void __launch_bounds__(VR_RAYCAST_THREADS, TEX ? VR_TEX_CTAS : VR_MIN_CTAS)
vr_raycast_kernel(const VrRaycastParams prm) {
    /* dynamic (ALPHA): the table, `copies` times (vr_march.cuh): 32 KB at most; what it does not take stays L1 cache */
    extern __shared__ float4 s_lut[];

    const VrGrid& g = prm.grid;
    const int lane = threadIdx.x & 31;
    __shared__ double s_minv[16];
    if (!RAYTAB && threadIdx.x < 16) s_minv[threadIdx.x] = prm.vs->Minv[threadIdx.x];
    const int copies = prm.lut_copies;
    if (MODE == VR_ALPHA) {
        for (int i = threadIdx.x; i < prm.lut.n * copies; i += blockDim.x) s_lut[i] = prm.lut.base[i / copies];
    }
    __syncthreads();
    if (prm.vs->singular) return;

    const int W = prm.vs->W, H = prm.vs->H;
    const int total = prm.vs->total_items;
    const float tau = prm.tau;
    LutView lut;
    lut.base = 0;
    lut.stride = 16u * (unsigned)copies;
    if (MODE == VR_ALPHA) {
        lut.base = (unsigned)__cvta_generic_to_shared(s_lut) + 16u * (unsigned)(lane & (copies - 1));
        asm volatile("" : "+r"(lut.base), "+r"(lut.stride)); /* two registers, not rebuilt per sample */
    }
    /* MIP may stop where the output saturates (vmax) or at the global maximum of the data when
     * it is known ("the maximum pixel value (defined by the global maximum of the data)") */
    const float mip_stop = fminf(prm.lut.vmax, prm.vs->data_max);
    unsigned long long nsamples = 0;

    /* one atomic per item; the next item is requested before the current one is processed */
    unsigned next = 0;
    if (lane == 0) next = atomicAdd(&prm.vs_rw->work_counter, 1u);
    next = __shfl_sync(FULL_MASK, next, 0);

    while (next < (unsigned)total) {
        const int item = (int)next;
        if (lane == 0) next = atomicAdd(&prm.vs_rw->work_counter, 1u);

        /* item -> (order position, tile) by binary search in the exclusive prefix */
        int lo_q = 0, hi_q = g.nbricks - 1;
        while (lo_q < hi_q) {
            const int mid = (lo_q + hi_q + 1) >> 1;
            if (__ldg(prm.item_prefix + mid) <= item) lo_q = mid;
            else hi_q = mid - 1;
        }
        const int b = __ldg(prm.order + lo_q);
        const int local = item - __ldg(prm.item_prefix + lo_q);
        const VrBrickView bvw = prm.bv[b];
        const int ty = local / bvw.tiles_x, tx = local - ty * bvw.tiles_x;
        const int pi = bvw.lx0 + tx * VR_TILE_W + (lane & 7);
        const int pj = bvw.ly0 + ty * VR_TILE_H + (lane >> 3);
        const bool in_launch = pi < bvw.lx1 && pj < bvw.ly1;
        const bool in_rect = in_launch && pi >= bvw.rx0 && pi < bvw.rx1 && pj >= bvw.ry0 && pj < bvw.ry1;

        int bc[3], blo[3], bhi[3], ext[3];
        vr_brick_coords(g, b, bc);
        vr_brick_core(g, bc, blo, bhi);
#pragma unroll
        for (int a = 0; a < 3; ++a) ext[a] = bhi[a] - blo[a] + 2 * g.ghost;
        const int slot_b = bvw.slot; /* = b unless the handle is a part (row f3) */
        const float* __restrict__ brick = prm.bricks + (long long)slot_b * g.slot;
        asm volatile("" : "+l"(brick)); /* keep the base in registers: do not rebuild it per load */

        RaySetup ray;
        ray.K = 0;
        ray.step = 1.0;
        int k_lo = 0, k_hi = 0;
        const long long ray_p = (long long)pj * W + pi;
        if (in_rect) {
            if (RAYTAB) ray_load<true>(prm.rays, prm.ray_plane, ray_p, prm.step, ray);
            else ray_setup(s_minv, W, H, pi, pj, g, prm.step, ray);
            brick_range(ray, g, bc, blo, bhi, k_lo, k_hi);
        }
        /* lattice samples: k in [k_lo, k_lat); samples k >= K-2 (whose interval may be clipped
         * by the exit point) are evaluated one by one in FP64 below */
        const int k_lat = min(k_hi, max(k_lo, ray.K - 2));
        int n = k_lat - k_lo;

        Accum acc;
        acc.r = (MODE == VR_MIP) ? -INFINITY : 0.0f;
        acc.g = acc.b = acc.a = 0.0f;
        Lattice L;
        long long D[3];
        float stepf = (float)ray.step; /* path length a lattice sample stands for */
        asm volatile("" : "+f"(stepf)); /* one register: not re-converted from the double in every loop trip */
        if (n > 0) {
            double s, w;
            sample_sw(ray, k_lo, s, w);
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
        /* texture arm: the sample position as the float32 texel coordinate of the brick's 3-D array, position of
         * step j = P0 + j * Df (one FFMA per axis; error < 1e-4 voxel, far below the filter's 2^-9 weight quantum) */
        cudaTextureObject_t tex = 0;
        float P0x = 0.0f, P0y = 0.0f, P0z = 0.0f, Dfx = 0.0f, Dfy = 0.0f, Dfz = 0.0f;
        const int n0 = n;
        bool use_tex = TEX && __ldg(prm.tex_nan + slot_b) == 0; /* warp-uniform: one brick per item */
        /* MIP through the arrays (below): eps bounds |filtered - exact| for every sample of this brick */
        float mip_eps = 0.0f, dec_a = 1.0f, dec_b = 0.0f;
        if (TEX && MODE == VR_MIP && use_tex) {
            const float2 bmm = __ldg(prm.brick_mm + b);
            /* + the float32 rounding of either filter, which scales with the magnitude, not the range */
            const float mag = fmaxf(fabsf(bmm.x), fabsf(bmm.y));
            mip_eps = (bmm.y - bmm.x) * prm.mip_range_eps + mag * prm.mip_mag_eps + prm.mip_abs_eps;
            if (prm.tex_byte) dec_a = bmm.y - bmm.x, dec_b = bmm.x; /* a byte fetch is (v - min) / (max - min) */
            /* a brick without finite voxels, or with voxels float16 texels cannot hold, keeps the hand-rolled loop */
            use_tex = mip_eps >= 0.0f && mip_eps < INFINITY && mag <= prm.mip_mag_max;
        }
        if (use_tex) {
            tex = __ldg(prm.tex + slot_b);
            const double h = 1.0 / 4294967296.0;
            P0x = (float)((double)L.q[0] * h + 0.5), P0y = (float)((double)L.q[1] * h + 0.5), P0z = (float)((double)L.q[2] * h + 0.5);
            Dfx = (float)((double)D[0] * h), Dfy = (float)((double)D[1] * h), Dfz = (float)((double)D[2] * h);
            /* six registers: not re-converted from the lattice in every loop trip */
            asm volatile("" : "+f"(P0x), "+f"(P0y), "+f"(P0z), "+f"(Dfx), "+f"(Dfy), "+f"(Dfz));
        }
        int stopped = (MODE == VR_ALPHA) ? !(acc.a < tau) : 0; /* int, not bool: no byte packing in the loop control */
        int active = n > 0 && !stopped;
        /* With step < 1 consecutive samples of a ray often fall into the same cell: the 8
         * voxels stay in registers and only the weights change (fewer L1 wavefronts, the
         * bound of densely sampled views). */
        Corners C;
        int pcx = INT_MIN, pcy = 0, pcz = 0;
        /* R19: samples based in a macro-cell the transfer function makes transparent are skipped (their
         * opacity is exactly 0): no voxel is fetched. The flag is looked up when the macro-cell changes. */
        const unsigned* __restrict__ cbits = (SKIP && MODE == VR_ALPHA) ? prm.cell_bits + (long long)slot_b * prm.cell_words : NULL;
        const float2* __restrict__ cmm = (SKIP && MODE == VR_MIP) ? prm.cell_mm + (long long)slot_b * (prm.nc[0] * prm.nc[1] * prm.nc[2]) : NULL;
        float pbound = INFINITY;
        int pm = -1;
        bool ptransp = false;
        /* Without macro-cell look-ups a lane's next positions do not depend on anything it loads: VR_TEX_DEPTH samples are
         * fetched back to back and then shaded in order, early termination tested between them as always (the values
         * fetched beyond a termination are dropped: at most VR_TEX_DEPTH - 1 per ray segment). The texture arm is bound by
         * the latency of its one fetch per sample at the 32 warps per SM its cache footprint allows (ncu: nothing above 40 %,
         * 12.8 warps per issue waiting on the scoreboard); this keeps VR_TEX_DEPTH fetches per warp in flight instead of one. */
        while (TEX && MODE == VR_ALPHA && !SKIP && use_tex && __any_sync(FULL_MASK, active)) {
            if (active) {
                const float kf = (float)(n0 - n);
                float vq[VR_TEX_DEPTH];
#pragma unroll
                for (int u = 0; u < VR_TEX_DEPTH; ++u) {
                    const float ku = kf + (float)u;
                    vq[u] = tex3D<float>(tex, fmaf(ku, Dfx, P0x), fmaf(ku, Dfy, P0y), fmaf(ku, Dfz, P0z));
                }
                bool by_hand = false; /* GUARD: the next sample of this lane is one for the hand-rolled sampler */
#pragma unroll
                for (int u = 0; u < VR_TEX_DEPTH; ++u) {
                    if (active && !by_hand) {
                        const float4 c = classify_alpha<true>(vq[u], lut, prm.lut);
                        if (GUARD && c.w > prm.tex_guard) {
                            by_hand = true; /* the rest of the batch is dropped and fetched again after it */
                        } else {
                            if (COUNT) nsamples += (vq[u] == vq[u]) ? 1 : 0;
                            blend_alpha(acc, vq[u], stepf, c);
                            stopped = !(acc.a < tau);
                            --n;
                            active = n > 0 && !stopped;
                        }
                    }
                }
                if (GUARD && by_hand) {
                    /* R20's guard (steps below one voxel): where the table's opacity nears 1 the opacity correction (1 - a)^w
                     * amplifies the filter's error without bound - this sample takes its value from the float32 store */
                    Lattice Lj;
                    const long long jj = (long long)(n0 - n);
                    Lj.q[0] = L.q[0] + D[0] * jj, Lj.q[1] = L.q[1] + D[1] * jj, Lj.q[2] = L.q[2] + D[2] * jj;
                    const float v = trilinear<LAY, PT, CLAMP, false>(brick, g, ext, Lj, prm.bitmap, (long long)slot_b * g.slot);
                    if (COUNT) nsamples += (v == v) ? 1 : 0;
                    shade_alpha<true>(acc, v, stepf, lut, prm.lut);
                    stopped = !(acc.a < tau);
                    --n;
                    active = n > 0 && !stopped;
                }
            }
        }
        while (TEX && MODE == VR_ALPHA && SKIP && use_tex && __any_sync(FULL_MASK, active)) {
            /* texture arm (built-in tri-linear interpolation): one TEX instead of 8 loads, the index
             * arithmetic and 7 FMA; the lattice is kept only where macro-cells are looked up (SKIP) */
            if (active) {
                int adv = 1;
                if (SKIP) {
                    const int cx = (int)(L.q[0] >> 32), cy = (int)(L.q[1] >> 32), cz = (int)(L.q[2] >> 32);
                    const int m = ((cz >> 3) * prm.nc[1] + (cy >> 3)) * prm.nc[0] + (cx >> 3);
                    if (m != pm) {
                        pm = m;
                        ptransp = (__ldg(cbits + (m >> 5)) >> (m & 31)) & 1u;
                    }
                    if (ptransp) adv = -leap_steps(L, D, n);
                }
                if (adv > 0) {
                    const float kf = (float)(n0 - n);
                    float v = tex3D<float>(tex, fmaf(kf, Dfx, P0x), fmaf(kf, Dfy, P0y), fmaf(kf, Dfz, P0z));
                    float4 c = classify_alpha<true>(v, lut, prm.lut);
                    if (GUARD && c.w > prm.tex_guard) { /* R20's guard, as above; the lattice is current here */
                        v = trilinear<LAY, PT, CLAMP, false>(brick, g, ext, L, prm.bitmap, (long long)slot_b * g.slot);
                        c = classify_alpha<true>(v, lut, prm.lut);
                    }
                    if (COUNT) nsamples += (v == v) ? 1 : 0;
                    blend_alpha(acc, v, stepf, c);
                    stopped = !(acc.a < tau);
                    if (SKIP) L.q[0] += D[0], L.q[1] += D[1], L.q[2] += D[2];
                } else {
                    adv = -adv;
                    L.q[0] += D[0] * adv, L.q[1] += D[1] * adv, L.q[2] += D[2] * adv;
                }
                n -= adv;
                active = n > 0 && !stopped;
            }
        }
        /* MIP through the arrays, EXACT (bit for bit the hand-rolled result): the filtered fetch serves as a bound, not as the
         * value. |filtered - exact| <= eps for every sample of the brick (the unit quantises the three weights to 8 fractional
         * bits: at most 3/256 of the largest difference between the 8 voxels, itself at most the brick's range; the float32 texel
         * coordinate adds < 3e-4 of it; eps = range / 64 + 2^-14 of the largest magnitude for the filters' own rounding - 2^-9 of it
         * when the texels are float16 (VR_SAMPLER_TEXTURE_HALF: rounding to float16 is within 2^-11 of a value, the rest is margin)),
         * so with hmax = the largest filtered value so far the segment's exact maximum is >= hmax - eps, and a sample whose
         * filtered value is below hmax - 2 eps cannot be it: only the others (the CANDIDATES: a few per cent on noise, the
         * records of the running maximum and their near misses) are evaluated by hand, in float32 from the tiled store, at the
         * same lattice position q0 + j D the hand-rolled loop reaches by repeated addition. A maximum does not depend on the
         * order of its operands. Candidates wait in a queue of VR_MIP_QUEUE (step, filtered value) pairs per lane; the warp
         * empties all queues when one is full, so the hand-rolled evaluations run with most lanes busy. */
        if (TEX && MODE == VR_MIP && use_tex) {
            int qj[VR_MIP_QUEUE];
            float qv[VR_MIP_QUEUE];
            int qn = 0;
            float hmax = -INFINITY;
            const float eps2 = mip_eps + mip_eps;
            const long long q0x = L.q[0], q0y = L.q[1], q0z = L.q[2];
            int j = 0; /* next lattice step of this lane */
            while (__any_sync(FULL_MASK, active || qn > 0)) {
                /* empty the queues: at the end of the segment, when a lane's queue is full, or when a lane may have
                 * reached the value at which MIP stops */
                const bool want = qn > 0 && (!active || qn == VR_MIP_QUEUE || hmax - mip_eps >= mip_stop);
                if (__any_sync(FULL_MASK, want)) {
#pragma unroll
                    for (int q = 0; q < VR_MIP_QUEUE; ++q) {
                        if (q < qn && qv[q] + mip_eps > acc.r && qv[q] >= hmax - eps2) {
                            Lattice Lj;
                            Lj.q[0] = q0x + D[0] * qj[q], Lj.q[1] = q0y + D[1] * qj[q], Lj.q[2] = q0z + D[2] * qj[q];
                            acc.r = fmaxf(acc.r, trilinear<LAY, PT, CLAMP, false>(brick, g, ext, Lj, prm.bitmap, (long long)slot_b * g.slot));
                        }
                    }
                    qn = 0;
                    stopped = acc.r >= mip_stop;
                    active = j < n0 && !stopped;
                }
                if (active) {
                    const float kf = (float)j;
                    float vq[VR_MIP_TEX_DEPTH];
#pragma unroll
                    for (int u = 0; u < VR_MIP_TEX_DEPTH; ++u) {
                        const float ku = kf + (float)u;
                        vq[u] = tex3D<float>(tex, fmaf(ku, Dfx, P0x), fmaf(ku, Dfy, P0y), fmaf(ku, Dfz, P0z));
                    }
#pragma unroll
                    for (int u = 0; u < VR_MIP_TEX_DEPTH; ++u) {
                        if (j < n0) {
                            const float v = fmaf(vq[u], dec_a, dec_b); /* float32 / float16 texels: v * 1 + 0, exact */
                            if (COUNT) ++nsamples; /* a brick seen through its array has no blanked voxel */
                            if (v >= hmax - eps2 && v + mip_eps > acc.r) {
                                if (qn < VR_MIP_QUEUE) {
#pragma unroll
                                    for (int q = 0; q < VR_MIP_QUEUE; ++q)
                                        if (q == qn) qj[q] = j, qv[q] = v;
                                    ++qn;
                                } else { /* no room (several candidates in one batch of fetches): evaluated at once */
                                    Lattice Lj;
                                    Lj.q[0] = q0x + D[0] * j, Lj.q[1] = q0y + D[1] * j, Lj.q[2] = q0z + D[2] * j;
                                    acc.r = fmaxf(acc.r, trilinear<LAY, PT, CLAMP, false>(brick, g, ext, Lj, prm.bitmap, (long long)slot_b * g.slot));
                                }
                            }
                            hmax = fmaxf(hmax, v);
                            ++j;
                        }
                    }
                    active = j < n0;
                }
            }
            n = 0;
            stopped = acc.r >= mip_stop;
        }
        while (!(TEX && use_tex) && __any_sync(FULL_MASK, active)) {
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
                        fetch8<LAY, PT, CLAMP, COUNT>(brick, g, ext, L, prm.bitmap, (long long)slot_b * g.slot, C);
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
                        shade_alpha<true>(acc, v, stepf, lut, prm.lut);
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
        /* the (at most two) samples next to the exit point */
        const int k_tail = max(k_lat, k_lo);
        if (__any_sync(FULL_MASK, k_tail < k_hi && !stopped)) {
#if VR_RECOMPUTE_TAIL
            if (k_tail < k_hi && !stopped) {
                if (RAYTAB) {
                    long long q = ray_p; /* an opaque copy: the ray is read again, not kept in registers through the loop */
                    asm volatile("" : "+l"(q));
                    ray_load<false>(prm.rays, prm.ray_plane, q, prm.step, ray);
                } else {
                    int qi = pi, qj = pj; /* opaque copies: the ray is rebuilt, not kept in registers */
                    asm volatile("" : "+r"(qi), "+r"(qj));
                    ray_setup(s_minv, W, H, qi, qj, g, prm.step, ray);
                }
            }
#endif
            for (int k = k_tail; k < k_hi && !stopped; ++k) {
                double s, w;
                if (!sample_sw(ray, k, s, w)) continue;
#pragma unroll
                for (int a = 0; a < 3; ++a) {
                    const double p = VR_FMA(s, ray.d[a], ray.o[a]);
                    L.q[a] = to_fixed(p - ((double)(blo[a] - g.ghost) + 0.5));
                }
                float v;
                if (TEX && MODE == VR_ALPHA && use_tex && prm.tex_only) { /* a released store has no float32 cells: the exit samples through the array too */
                    const double h = 1.0 / 4294967296.0;
                    v = tex3D<float>(tex, (float)((double)L.q[0] * h + 0.5), (float)((double)L.q[1] * h + 0.5), (float)((double)L.q[2] * h + 0.5));
                } else {
                    v = trilinear<LAY, PT, CLAMP, COUNT>(brick, g, ext, L, prm.bitmap, (long long)slot_b * g.slot);
                }
                if (COUNT) nsamples += (v == v) ? 1 : 0;
                if (MODE == VR_MIP) {
                    acc.r = fmaxf(acc.r, v);
                    stopped = acc.r >= mip_stop;
                } else {
                    shade_alpha<true>(acc, v, (float)w, lut, prm.lut);
                    stopped = !(acc.a < tau);
                }
            }
        }

        /* row a8: one sub-image pixel per pixel of the launch rectangle */
        if (in_launch) {
            const long long off = bvw.sub_offset + (long long)(pj - bvw.ly0) * (bvw.lx1 - bvw.lx0) + (pi - bvw.lx0);
            if (MODE == VR_ALPHA) reinterpret_cast<float4*>(prm.sub)[off] = make_float4(acc.r, acc.g, acc.b, acc.a);
            else reinterpret_cast<float*>(prm.sub)[off] = acc.r;
        }
        next = __shfl_sync(FULL_MASK, next, 0);
    }
    if (COUNT) {
        for (int o = 16; o > 0; o >>= 1) nsamples += __shfl_xor_sync(FULL_MASK, nsamples, o);
        if (lane == 0 && nsamples) atomicAdd(&prm.vs_rw->samples, nsamples);
    }
}

/* ------------------------------------------------------------------------------------------ */
/* Persistent grid: resident CTAs per SM (for this instance and its shared memory) x SMs,
 * but no more CTAs than there are groups of 8 work items. */
template <int MODE, int LAY, int PT, bool CLAMP, bool COUNT, bool SKIP, bool TEX, bool RAYTAB, bool GUARD>
static cudaError_t launch_instance(const VrRaycastParams& p0, long long items, bool sparse, cudaStream_t st);

template <int MODE, int LAY, int PT, bool CLAMP, bool COUNT, bool SKIP = false, bool TEX = false>
static cudaError_t launch_variant(const VrRaycastParams& p, long long items, bool sparse, cudaStream_t st) {
    if constexpr (TEX && MODE == VR_ALPHA) { /* R20's guard is compiled into the instances that need it only (steps below one voxel) */
        if (p.tex_guard <= 1.0f)
            return p.rays ? launch_instance<MODE, LAY, PT, CLAMP, COUNT, SKIP, TEX, true, true>(p, items, sparse, st)
                          : launch_instance<MODE, LAY, PT, CLAMP, COUNT, SKIP, TEX, false, true>(p, items, sparse, st);
    }
    return p.rays ? launch_instance<MODE, LAY, PT, CLAMP, COUNT, SKIP, TEX, true, false>(p, items, sparse, st)
                  : launch_instance<MODE, LAY, PT, CLAMP, COUNT, SKIP, TEX, false, false>(p, items, sparse, st);
}

template <int MODE, int LAY, int PT, bool CLAMP, bool COUNT, bool SKIP, bool TEX, bool RAYTAB, bool GUARD>
static cudaError_t launch_instance(const VrRaycastParams& p0, long long items, bool sparse, cudaStream_t st) {
    VrRaycastParams p = p0;
    p.lut_copies = vr_lut_copies(p.lut.n, sparse);
    if (TEX && p.lut_copies > VR_TEX_COPIES) p.lut_copies = VR_TEX_COPIES;
    const size_t smem = MODE == VR_ALPHA ? sizeof(float4) * (size_t)p.lut.n * p.lut_copies : 0;
    /* asked of the runtime at every launch (a few microseconds): the current device's SM count and this instance's
     * residency with this much shared memory - no process-wide cache to go stale across devices or threads */
    int dev = 0, sms = 0, cached_per_sm = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (e == cudaSuccess)
        e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&cached_per_sm, vr_raycast_kernel<MODE, LAY, PT, CLAMP, COUNT, SKIP, TEX, RAYTAB, GUARD>,
                                                          VR_RAYCAST_THREADS, smem);
    if (e != cudaSuccess) return e;
    if (cached_per_sm < 1) return cudaErrorLaunchOutOfResources;
    /* Sparse MIP frames (several voxels per pixel: every load is a DRAM line of its own) run faster with two
     * resident CTAs per SM than with three - the lighter MIP loop keeps more lines in flight than L1/L2 hold
     * (c3: 14.5 -> 12.3 ms); dense frames and ALPHA want all three. */
    int per_sm = (MODE == VR_MIP && sparse && cached_per_sm > 2) ? 2 : cached_per_sm;
#ifdef VR_EXP_SPARSE_TEX_PER_SM /* experiment knob (profiles/r2_c3_experiments.md): resident CTAs of the texture arm on sparse views */
    if (TEX && sparse && per_sm > VR_EXP_SPARSE_TEX_PER_SM) per_sm = VR_EXP_SPARSE_TEX_PER_SM;
#endif
    long long ctas = (long long)sms * per_sm;
    const long long want = (items + (VR_RAYCAST_THREADS / 32) - 1) / (VR_RAYCAST_THREADS / 32);
    if (ctas > want) ctas = want < 1 ? 1 : want;
    vr_raycast_kernel<MODE, LAY, PT, CLAMP, COUNT, SKIP, TEX, RAYTAB, GUARD><<<(int)ctas, VR_RAYCAST_THREADS, smem, st>>>(p);
    return cudaGetLastError();
}

static bool is_tile442(const VrGrid& g) {
    return g.layout == VR_LAYOUT_TILED && g.tl[0] == 2 && g.tl[1] == 2 && g.tl[2] == 1 && g.ml[0] == 0 && g.ml[1] == 0 &&
           g.ml[2] == 0;
}

template <int MODE, bool COUNT>
static cudaError_t launch_mode(const VrRaycastParams& p, long long ctas, bool sparse, cudaStream_t st) {
    const bool clamp = p.grid.ghost == 0;
    if (p.grid.layout == VR_LAYOUT_LINEAR) {
        if (clamp) return launch_variant<MODE, LAY_LINEAR, 0, true, COUNT>(p, ctas, sparse, st);
        switch (p.grid.P) {
            case 258: return launch_variant<MODE, LAY_LINEAR, 258, false, COUNT>(p, ctas, sparse, st);
            case 514: return launch_variant<MODE, LAY_LINEAR, 514, false, COUNT>(p, ctas, sparse, st);
            default: return launch_variant<MODE, LAY_LINEAR, 0, false, COUNT>(p, ctas, sparse, st);
        }
    }
    if (is_tile442(p.grid) && p.tex != NULL && MODE == VR_ALPHA && p.bitmap == NULL) {
        /* texture arm (vr_set_sampler), VR_ALPHA values; the touched-cells bitmap is the hand-rolled path's */
        if (!clamp && p.cell_bits != NULL) return launch_variant<VR_ALPHA, LAY_TILE442, 0, false, COUNT, true, true>(p, ctas, sparse, st);
        return clamp ? launch_variant<VR_ALPHA, LAY_TILE442, 0, true, COUNT, false, true>(p, ctas, sparse, st)
                     : launch_variant<VR_ALPHA, LAY_TILE442, 0, false, COUNT, false, true>(p, ctas, sparse, st);
    }
    if (is_tile442(p.grid) && p.tex != NULL && MODE == VR_MIP && p.bitmap == NULL && p.brick_mm != NULL && p.cell_mm == NULL) {
        /* texture arm, MIP: the arrays as an exact filter in front of the hand-rolled sampler (the MIP loop of the kernel) */
        return clamp ? launch_variant<VR_MIP, LAY_TILE442, 0, true, COUNT, false, true>(p, ctas, sparse, st)
                     : launch_variant<VR_MIP, LAY_TILE442, 0, false, COUNT, false, true>(p, ctas, sparse, st);
    }
    if (is_tile442(p.grid)) {
        /* R19: macro-cell skipping - ALPHA when the transfer function has a transparent range, MIP when the cube has empty space */
        if (!clamp && (MODE == VR_ALPHA ? p.cell_bits != NULL : p.cell_mm != NULL))
            return launch_variant<MODE, LAY_TILE442, 0, false, COUNT, true>(p, ctas, sparse, st);
        return clamp ? launch_variant<MODE, LAY_TILE442, 0, true, COUNT>(p, ctas, sparse, st)
                     : launch_variant<MODE, LAY_TILE442, 0, false, COUNT>(p, ctas, sparse, st);
    }
    return clamp ? launch_variant<MODE, LAY_GENERIC, 0, true, COUNT>(p, ctas, sparse, st)
                 : launch_variant<MODE, LAY_GENERIC, 0, false, COUNT>(p, ctas, sparse, st);
}

cudaError_t vr_launch_raycast(const VrRaycastParams& p, long long ctas, bool count, bool sparse, cudaStream_t st) {
    if (p.mode == VR_ALPHA) return count ? launch_mode<VR_ALPHA, true>(p, ctas, sparse, st) : launch_mode<VR_ALPHA, false>(p, ctas, sparse, st);
    return count ? launch_mode<VR_MIP, true>(p, ctas, sparse, st) : launch_mode<VR_MIP, false>(p, ctas, sparse, st);
}
