/*
 * vr_setup.cu -- per-view set-up and device-side visibility sort (SURVEY.md sec. 8(a) rows
 * a2, a3). One CTA per frame, no host involvement:
 *   1. M = proj*view, its inverse, the homogeneous eye (vr_view.cuh).
 *   2. Per-axis slab ranks by distance from the eye (perspective) or by the sign of the view
 *      direction (orthographic); brick key = (rank_z, rank_y, rank_x) lexicographic. The
 *      ranks are permutations, so the key IS the brick's position in the front-to-back
 *      order: the sort is a direct scatter, exact and deterministic (R9). PAPER.md:53 names
 *      depth sorting as one of the tasks done in CUDA; :174 needs the order for `over`.
 *   3. Per brick: rendering rectangle = bounding box of its 8 projected vertices
 *      (Fig. 4 :168), launch rectangle on the 8x4 tile grid, tile counts.
 *   4. Exclusive scans, in visibility order, of the tile counts (work list of the persistent
 *      ray-cast kernel) and of the sub-image sizes (scratch offsets); compositing table.
 *   5. Row f1: with the per-brick data range known (vr_minmax.cu), ALPHA frames skip the bricks
 *      the transfer function makes transparent (R16: every table entry the brick's values can
 *      interpolate between has alpha 0, entry range widened by -1/+2): no work items, no
 *      sub-image, an empty compositing rectangle. Exact: such a brick contributes zeros.
 *   6. Row f3: a part handle gives an empty rectangle to every brick outside its box; what it renders is the
 *      partial frame of its own bricks, in the global visibility order.
 */
#include "vr_view.cuh"

#define SETUP_THREADS 256

struct SetupShared {
    double M[16];
    int rank[3][VR_MAX_AXIS_BRICKS];
    int warp_items[SETUP_THREADS / 32];
    long long warp_pix[SETUP_THREADS / 32];
    int carry_items;
    long long carry_pix;
    int ortho;
    double eye[3];
    int culled;
    unsigned short nz_prefix[VR_MAX_LUT + 1]; /* nz_prefix[i] = entries < i with alpha != 0 */
    /* grids of up to SETUP_THREADS bricks keep their views and order here between the passes (the global
     * copies are written once, complete, at the end): no global round trips inside the kernel */
    VrBrickView bv[SETUP_THREADS];
    int order[SETUP_THREADS];
    int bound[4]; /* union of the non-empty rendering rectangles */
};

__global__ void __launch_bounds__(SETUP_THREADS)
vr_setup_kernel(VrGrid grid, VrMatrices mats, int W, int H, int mode, long long sub_capacity_px,
                unsigned long long sub_base, VrViewState* __restrict__ vs, VrBrickView* __restrict__ bv,
                int* __restrict__ order, int* __restrict__ item_prefix, VrCompLayer* __restrict__ layers,
                const float2* __restrict__ range, VrLut lut, int* __restrict__ overflow_flag) {
    __shared__ SetupShared sh;
    const int tid = threadIdx.x;
    const bool small = grid.nbricks <= SETUP_THREADS;
    const bool cull = range != NULL && mode == VR_ALPHA && lut.base != NULL;
    /* the global reads the passes below wait for are issued first, ahead of the matrix inversion */
    float2 mm0 = make_float2(0.0f, 0.0f);
    if (cull && tid < grid.nbricks) mm0 = range[tid];
    if (tid == 64) vs->data_max = range ? range[grid.nbricks].y : INFINITY;

    /* warp 0: M = P*V and its Gauss-Jordan inverse with one lane per entry of the augmented 4 x 8 matrix - the
     * operations of vr_view_setup (vr_view.cuh), entry by entry and in the same order, so the same bits (R9, R10) */
    if (tid < 32) {
        const unsigned FULL = 0xffffffffu;
        const int r = tid >> 3, c = tid & 7;
        double m = 0.0;
        if (tid < 16) { /* entry (row tid & 3, column tid >> 2) of M, column-major */
            const int mr = tid & 3, mc = tid >> 2;
            for (int k = 0; k < 4; ++k) m = VR_ADD(m, VR_MUL((double)mats.proj[k * 4 + mr], (double)mats.view[mc * 4 + k]));
            sh.M[tid] = m;
            vs->M[tid] = m;
        }
        /* a = [M | I](r, c): M(r, c) lives in lane c * 4 + r */
        double a = __shfl_sync(FULL, m, (c & 3) * 4 + r);
        if (c >= 4) a = (r == c - 4) ? 1.0 : 0.0;
        int bad = 0;
        for (int col = 0; col < 4; ++col) {
            int piv = col;
            double best = fabs(__shfl_sync(FULL, a, col * 8 + col));
            for (int rr = col + 1; rr < 4; ++rr) {
                const double v = fabs(__shfl_sync(FULL, a, rr * 8 + col));
                if (v > best) {
                    best = v;
                    piv = rr;
                }
            }
            if (best == 0.0) {
                bad = 1;
                break;
            }
            const double from_piv = __shfl_sync(FULL, a, piv * 8 + c), from_col = __shfl_sync(FULL, a, col * 8 + c);
            if (piv != col) {
                if (r == col) a = from_piv;
                else if (r == piv) a = from_col;
            }
            const double d = __shfl_sync(FULL, a, col * 8 + col);
            if (r == col) a = VR_DIV(a, d);
            const double f = __shfl_sync(FULL, a, r * 8 + col), pc = __shfl_sync(FULL, a, col * 8 + c);
            if (r != col && f != 0.0) a = VR_SUB(a, VR_MUL(f, pc));
        }
        if (__any_sync(FULL, c >= 4 && !isfinite(a))) bad = 1;
        if (c >= 4) vs->Minv[(c - 4) * 4 + r] = a;
        /* homogeneous eye = third column of Minv: lanes r * 8 + 6 */
        const double c0 = __shfl_sync(FULL, a, 6), c1 = __shfl_sync(FULL, a, 14), c2 = __shfl_sync(FULL, a, 22),
                     c3 = __shfl_sync(FULL, a, 30);
        if (tid == 0) {
            int ortho = 0;
            if (!bad) {
                const double mag = VR_ADD(VR_ADD(fabs(c0), fabs(c1)), fabs(c2));
                if (fabs(c3) < VR_MUL(1e-9, mag)) {
                    ortho = 1;
                    sh.eye[0] = c0; sh.eye[1] = c1; sh.eye[2] = c2;
                } else {
                    sh.eye[0] = VR_DIV(c0, c3); sh.eye[1] = VR_DIV(c1, c3); sh.eye[2] = VR_DIV(c2, c3);
                }
            } else {
                sh.eye[0] = sh.eye[1] = sh.eye[2] = 0.0;
            }
            sh.ortho = ortho;
            for (int i = 0; i < 3; ++i) vs->eye[i] = sh.eye[i];
            vs->ortho = ortho;
            vs->singular = bad;
            vs->W = W;
            vs->H = H;
            vs->work_counter = 0u;
            vs->samples = 0ull;
            sh.carry_items = 0;
            sh.carry_pix = 0;
            sh.culled = 0;
            sh.bound[0] = W; sh.bound[1] = H; sh.bound[2] = 0; sh.bound[3] = 0;
        }
    }
    if (cull) { /* block scan of the alpha != 0 flags: 4 consecutive entries per thread (n <= VR_MAX_LUT = 4 * 256) */
        int f[4], t = 0;
        for (int j = 0; j < 4; ++j) {
            const int i = 4 * tid + j;
            f[j] = (i < lut.n && lut.base[i].w != 0.0f) ? 1 : 0;
            t += f[j];
        }
        int incl = t;
        for (int o = 1; o < 32; o <<= 1) {
            const int u = __shfl_up_sync(0xffffffffu, incl, o);
            if ((tid & 31) >= o) incl += u;
        }
        if ((tid & 31) == 31) sh.warp_items[tid >> 5] = incl;
        __syncthreads();
        int run = incl - t;
        for (int w = 0; w < (tid >> 5); ++w) run += sh.warp_items[w];
        if (tid == 0) sh.nz_prefix[0] = 0;
        for (int j = 0; j < 4; ++j) {
            const int i = 4 * tid + j;
            run += f[j];
            if (i < lut.n) sh.nz_prefix[i + 1] = (unsigned short)run;
        }
    }
    __syncthreads();

    /* per-axis ranks (R9) */
    for (int a = 0; a < 3; ++a) {
        const int n = grid.g[a];
        for (int i = tid; i < n; i += SETUP_THREADS) {
            int r;
            if (sh.ortho) {
                r = (sh.eye[a] >= 0.0) ? i : (n - 1 - i);
            } else {
                const double e = sh.eye[a];
                double lo = (double)i * (double)grid.brick, hi = lo + (double)grid.brick;
                if (hi > (double)grid.n[a]) hi = (double)grid.n[a];
                const double di = (e < lo) ? VR_SUB(lo, e) : ((e > hi) ? VR_SUB(e, hi) : 0.0);
                r = 0;
                for (int j = 0; j < n; ++j) {
                    double lj = (double)j * (double)grid.brick, hj = lj + (double)grid.brick;
                    if (hj > (double)grid.n[a]) hj = (double)grid.n[a];
                    const double dj = (e < lj) ? VR_SUB(lj, e) : ((e > hj) ? VR_SUB(e, hj) : 0.0);
                    if (dj < di || (dj == di && j < i)) ++r;
                }
            }
            sh.rank[a][i] = r;
        }
    }
    __syncthreads();

    /* per brick: order position, rectangles */
    for (int b = tid; b < grid.nbricks; b += SETUP_THREADS) {
        int bc[3], lo[3], hi[3], r[4], l[4];
        vr_brick_coords(grid, b, bc);
        vr_brick_core(grid, bc, lo, hi);
        const int key = (sh.rank[2][bc[2]] * grid.g[1] + sh.rank[1][bc[1]]) * grid.g[0] + sh.rank[0][bc[0]];
        if (small) sh.order[key] = b;
        order[key] = b;
        vr_rect_of_box(sh.M, lo, hi, W, H, r);
        if (vr_slot_index(grid, b) < 0) r[2] = r[0]; /* row f3: another part holds this brick */
        if (cull) { /* R16, float32 as the ray-cast kernel classifies */
            const float2 mm = (b == tid) ? mm0 : range[b];
            const float ulo = __saturatef(__fmul_rn(__fsub_rn(mm.x, lut.vmin), lut.inv_range));
            const float uhi = __saturatef(__fmul_rn(__fsub_rn(mm.y, lut.vmin), lut.inv_range));
            const int i0 = max(min((int)__fmul_rn(ulo, lut.scale), lut.nm2) - 1, 0);
            const int i1 = min(min((int)__fmul_rn(uhi, lut.scale), lut.nm2) + 2, lut.n - 1);
            if (sh.nz_prefix[i1 + 1] == sh.nz_prefix[i0] && r[2] > r[0] && r[3] > r[1]) {
                r[2] = r[0]; /* empty rectangle: nothing to cast, nothing to composite */
                atomicAdd(&sh.culled, 1);
            }
        }
        if (r[2] > r[0] && r[3] > r[1]) {
            atomicMin(&sh.bound[0], r[0]);
            atomicMin(&sh.bound[1], r[1]);
            atomicMax(&sh.bound[2], r[2]);
            atomicMax(&sh.bound[3], r[3]);
        }
        vr_launch_rect(r, W, H, l);
        VrBrickView v;
        v.rx0 = r[0]; v.ry0 = r[1]; v.rx1 = r[2]; v.ry1 = r[3];
        v.lx0 = l[0]; v.ly0 = l[1]; v.lx1 = l[2]; v.ly1 = l[3];
        v.tiles_x = (l[2] - l[0] + VR_TILE_W - 1) / VR_TILE_W;
        v.tiles_y = (l[3] - l[1] + VR_TILE_H - 1) / VR_TILE_H;
        v.order_pos = key;
        v.slot = vr_slot_index(grid, b);
        v.sub_offset = 0;
        *(small ? &sh.bv[b] : &bv[b]) = v;
    }
    __syncthreads();
    __threadfence_block();

    /* exclusive scans over order positions, 256 at a time with a running carry */
    const int lane = tid & 31, wid = tid >> 5;
    for (int q0 = 0; q0 < grid.nbricks; q0 += SETUP_THREADS) {
        const int q = q0 + tid;
        int items = 0;
        long long pix = 0;
        int b = -1;
        if (q < grid.nbricks) {
            b = small ? sh.order[q] : order[q];
            const VrBrickView* v = small ? &sh.bv[b] : &bv[b];
            items = v->tiles_x * v->tiles_y;
            pix = (long long)(v->lx1 - v->lx0) * (long long)(v->ly1 - v->ly0);
        }
        int si = items;
        long long sp = pix;
        for (int o = 1; o < 32; o <<= 1) {
            const int ti = __shfl_up_sync(0xffffffffu, si, o);
            const long long tp = __shfl_up_sync(0xffffffffu, sp, o);
            if (lane >= o) {
                si += ti;
                sp += tp;
            }
        }
        if (lane == 31) {
            sh.warp_items[wid] = si;
            sh.warp_pix[wid] = sp;
        }
        __syncthreads();
        int bi = sh.carry_items;
        long long bp = sh.carry_pix;
        for (int w = 0; w < wid; ++w) {
            bi += sh.warp_items[w];
            bp += sh.warp_pix[w];
        }
        if (q < grid.nbricks) {
            item_prefix[q] = bi + si - items;
            if (small) sh.bv[b].sub_offset = bp + sp - pix;
            else bv[b].sub_offset = bp + sp - pix;
        }
        __syncthreads();
        if (tid == SETUP_THREADS - 1) {
            sh.carry_items = bi + si;
            sh.carry_pix = bp + sp;
        }
        __syncthreads();
    }

    if (tid == 0) {
        const int over = sh.carry_pix > sub_capacity_px;
        item_prefix[grid.nbricks] = sh.carry_items;
        vs->total_items = over ? 0 : sh.carry_items;
        vs->total_sub_pixels = sh.carry_pix;
        vs->overflow = over;
        if (over && overflow_flag) *overflow_flag = 1; /* mapped host memory: the host sees it without a copy */
        vs->culled = sh.culled;
        const bool none = sh.bound[2] <= sh.bound[0] || sh.bound[3] <= sh.bound[1];
        for (int i = 0; i < 4; ++i) vs->bound[i] = none ? 0 : sh.bound[i];
    }
    __syncthreads();

    /* compositing table: one layer per brick */
    const unsigned long long px_bytes = (mode == VR_ALPHA) ? 16ull : 4ull;
    const bool over = sh.carry_pix > sub_capacity_px;
    for (int b = tid; b < grid.nbricks; b += SETUP_THREADS) {
        const VrBrickView v = *(small ? &sh.bv[b] : &bv[b]);
        if (small) bv[b] = v;
        VrCompLayer L;
        L.x0 = v.rx0; L.y0 = v.ry0; L.x1 = over ? v.rx0 : v.rx1; L.y1 = v.ry1;
        L.sx0 = v.lx0; L.sy0 = v.ly0;
        L.pitch = v.lx1 - v.lx0;
        L.pad = 0;
        L.addr = sub_base + (unsigned long long)v.sub_offset * px_bytes;
        layers[b] = L;
    }
}

cudaError_t vr_launch_setup(const VrGrid& grid, const VrMatrices& mats, int W, int H, int mode, long long sub_capacity_px,
                            void* sub_base, VrViewState* vs, VrBrickView* bv, int* order, int* item_prefix,
                            VrCompLayer* layers, const float2* range, const VrLut& lut, int* overflow_flag, cudaStream_t st) {
    vr_setup_kernel<<<1, SETUP_THREADS, 0, st>>>(grid, mats, W, H, mode, sub_capacity_px,
                                                 (unsigned long long)(uintptr_t)sub_base, vs, bv, order, item_prefix, layers,
                                                 range, lut, overflow_flag);
    return cudaGetLastError();
}

/* Host mirror: is proj*view invertible, and how much scratch does this view need. Used for
 * argument validation and scratch sizing only; the frame itself uses the kernel's values. */
int vr_host_view_check(const VrGrid& grid, const float* view, const float* proj, int W, int H, long long* sub_pixels,
                       long long* items) {
    double M[16], Minv[16], eye[3];
    int ortho;
    if (vr_view_setup(view, proj, M, Minv, eye, &ortho)) return 1;
    long long pix = 0, it = 0;
    for (int b = 0; b < grid.nbricks; ++b) {
        int bc[3], lo[3], hi[3], r[4], l[4];
        if (vr_slot_index(grid, b) < 0) continue; /* a part renders its own bricks only */
        vr_brick_coords(grid, b, bc);
        vr_brick_core(grid, bc, lo, hi);
        vr_rect_of_box(M, lo, hi, W, H, r);
        /* one pixel of slack per side in case host and device round a vertex differently */
        if (r[2] > r[0] && r[3] > r[1]) {
            r[0] = r[0] > 0 ? r[0] - 1 : 0;
            r[1] = r[1] > 0 ? r[1] - 1 : 0;
            r[2] = r[2] < W ? r[2] + 1 : W;
            r[3] = r[3] < H ? r[3] + 1 : H;
        } else {
            r[0] = 0; r[1] = 0; r[2] = 2 < W ? 2 : W; r[3] = 2 < H ? 2 : H;
        }
        vr_launch_rect(r, W, H, l);
        pix += (long long)(l[2] - l[0]) * (l[3] - l[1]);
        it += (long long)((l[2] - l[0] + VR_TILE_W - 1) / VR_TILE_W) * ((l[3] - l[1] + VR_TILE_H - 1) / VR_TILE_H);
    }
    *sub_pixels = pix;
    *items = it;
    return 0;
}

/* Row f3: a rectangle that contains the rendering rectangle of every brick the handle holds (the union of
 * the per-brick rectangles of PAPER.md:150, one pixel of slack per side as above): the part of the frame a
 * part's partial image can be non-blank in, which is what travels in the exchange. */
int vr_host_part_rect(const VrGrid& grid, const float* view, const float* proj, int W, int H, int rect[4]) {
    double M[16], Minv[16], eye[3];
    int ortho;
    if (vr_view_setup(view, proj, M, Minv, eye, &ortho)) return 1;
    int u[4] = {W, H, 0, 0};
    for (int b = 0; b < grid.nbricks; ++b) {
        int bc[3], lo[3], hi[3], r[4];
        if (vr_slot_index(grid, b) < 0) continue;
        vr_brick_coords(grid, b, bc);
        vr_brick_core(grid, bc, lo, hi);
        vr_rect_of_box(M, lo, hi, W, H, r);
        if (r[2] <= r[0] || r[3] <= r[1]) continue;
        r[0] = r[0] > 0 ? r[0] - 1 : 0;
        r[1] = r[1] > 0 ? r[1] - 1 : 0;
        r[2] = r[2] < W ? r[2] + 1 : W;
        r[3] = r[3] < H ? r[3] + 1 : H;
        if (r[0] < u[0]) u[0] = r[0];
        if (r[1] < u[1]) u[1] = r[1];
        if (r[2] > u[2]) u[2] = r[2];
        if (r[3] > u[3]) u[3] = r[3];
    }
    if (u[2] <= u[0] || u[3] <= u[1]) u[0] = u[1] = u[2] = u[3] = 0;
    for (int i = 0; i < 4; ++i) rect[i] = u[i];
    return 0;
}
