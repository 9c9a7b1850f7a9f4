/*
 * vr_synth_cpu.c -- host side of the seeded input generator (see vr_synth.h).
 *
 * Builds the source catalogue (positions, peaks, widths, 1-D Gaussian profile
 * tables, cell -> source lists) from the seed and evaluates voxels on the CPU.
 * The CUDA twin (vr_synth_cuda.cu) uploads the SAME tables and runs the SAME
 * vs_voxel(), so both produce bit-identical cubes.
 *
 * Recipe: i.i.d. N(0,1) noise; N_src sources with
 * centre uniform in the volume, peak U[3,10] sigma, FWHM_x, FWHM_y U[3,8] voxels,
 * FWHM_z U[2,20] channels, axis-aligned Gaussian, sigma = FWHM/2.3548, cut at
 * +-5 sigma; optional ramp*(z+1/2)/nz along the spectral axis.
 *
 * Build: gcc -O2 -ffp-contract=off -fopenmp -shared -fPIC (synth/build.py).
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#include "vr_synth.h"

static double u01(uint64_t seed, uint64_t stream, uint64_t i) {
    uint64_t h = vs_hash2(seed ^ (0xA5A5A5A5ULL + stream * 0x100000001B3ULL), i);
    return ((double)(h >> 11) + 0.5) * (1.0 / 9007199254740992.0);
}

static int64_t clampi(int64_t v, int64_t lo, int64_t hi) { return v < lo ? lo : (v > hi ? hi : v); }

vs_cube* vs_cube_create_kind(uint64_t seed, int64_t nx, int64_t ny, int64_t nz, int32_t nsrc, double ramp, int32_t kind);

vs_cube* vs_cube_create(uint64_t seed, int64_t nx, int64_t ny, int64_t nz, int32_t nsrc, double ramp) {
    return vs_cube_create_kind(seed, nx, ny, nz, nsrc, ramp, VS_SPECTRAL);
}

/* kind VS_NBODY: density-cube stand-in (Table 1 "Nbody"): zero background, nsrc halos with
 * log-uniform central density 0.5..30 and FWHM 4..32 voxels per axis, truncated at 5 sigma. */
vs_cube* vs_cube_create_kind(uint64_t seed, int64_t nx, int64_t ny, int64_t nz, int32_t nsrc, double ramp, int32_t kind) {
    if (nx <= 0 || ny <= 0 || nz <= 0 || nsrc < 0 || (kind != VS_SPECTRAL && kind != VS_NBODY)) return NULL;
    vs_cube* c = (vs_cube*)calloc(1, sizeof(vs_cube));
    c->seed = seed; c->nx = nx; c->ny = ny; c->nz = nz; c->ramp = ramp; c->nsrc = nsrc; c->kind = kind;
    c->cgx = (int32_t)((nx + VS_CELL - 1) / VS_CELL);
    c->cgy = (int32_t)((ny + VS_CELL - 1) / VS_CELL);
    c->cgz = (int32_t)((nz + VS_CELL - 1) / VS_CELL);
    int64_t ncell = (int64_t)c->cgx * c->cgy * c->cgz;
    int32_t* start = (int32_t*)calloc((size_t)ncell + 1, sizeof(int32_t));
    size_t ns = nsrc > 0 ? (size_t)nsrc : 1;
    int32_t *x0 = malloc(ns * 4), *y0 = malloc(ns * 4), *z0 = malloc(ns * 4);
    int32_t *lx = malloc(ns * 4), *ly = malloc(ns * 4), *lz = malloc(ns * 4);
    int32_t *ox = malloc(ns * 4), *oy = malloc(ns * 4), *oz = malloc(ns * 4);
    float* peak = malloc(ns * 4);
    size_t nprof = 0, cap = 1024;
    float* prof = malloc(cap * sizeof(float));

    const int64_t dims[3] = {nx, ny, nz};
    for (int32_t s = 0; s < nsrc; ++s) {
        double ctr[3], sig[3];
        ctr[0] = u01(seed, 1, s) * (double)nx;
        ctr[1] = u01(seed, 2, s) * (double)ny;
        ctr[2] = u01(seed, 3, s) * (double)nz;
        peak[s] = (float)(3.0 + 7.0 * u01(seed, 4, s));
        sig[0] = (3.0 + 5.0 * u01(seed, 5, s)) / 2.3548;
        sig[1] = (3.0 + 5.0 * u01(seed, 6, s)) / 2.3548;
        sig[2] = (2.0 + 18.0 * u01(seed, 7, s)) / 2.3548;
        if (kind == VS_NBODY) {
            peak[s] = (float)(0.5 * exp(u01(seed, 4, s) * log(60.0)));
            for (int a = 0; a < 3; ++a) sig[a] = (4.0 + 28.0 * u01(seed, 5 + a, s)) / 2.3548;
        }
        int32_t org[3], len[3], off[3];
        for (int a = 0; a < 3; ++a) {
            int64_t lo = clampi((int64_t)floor(ctr[a] - 5.0 * sig[a]), 0, dims[a] - 1);
            int64_t hi = clampi((int64_t)ceil(ctr[a] + 5.0 * sig[a]), lo + 1, dims[a]);
            org[a] = (int32_t)lo; len[a] = (int32_t)(hi - lo); off[a] = (int32_t)nprof;
            if (nprof + (size_t)len[a] > cap) {
                while (nprof + (size_t)len[a] > cap) cap *= 2;
                prof = realloc(prof, cap * sizeof(float));
            }
            for (int32_t i = 0; i < len[a]; ++i) {
                double t = ((double)(lo + i) + 0.5 - ctr[a]) / sig[a];
                prof[nprof++] = (float)exp(-0.5 * t * t);
            }
        }
        x0[s] = org[0]; y0[s] = org[1]; z0[s] = org[2];
        lx[s] = len[0]; ly[s] = len[1]; lz[s] = len[2];
        ox[s] = off[0]; oy[s] = off[1]; oz[s] = off[2];
    }
    /* cell lists: count, prefix, fill in ascending source order */
    for (int pass = 0; pass < 2; ++pass) {
        int32_t* fillpos = NULL;
        int32_t* items = NULL;
        if (pass == 1) {
            int32_t run = 0;
            for (int64_t i = 0; i < ncell; ++i) { int32_t n = start[i]; start[i] = run; run += n; }
            start[ncell] = run;
            items = malloc((run > 0 ? (size_t)run : 1) * sizeof(int32_t));
            fillpos = malloc((size_t)(ncell > 0 ? ncell : 1) * sizeof(int32_t));
            memcpy(fillpos, start, (size_t)ncell * sizeof(int32_t));
            c->cell_items = items;
        }
        for (int32_t s = 0; s < nsrc; ++s) {
            int32_t cx0 = x0[s] / VS_CELL, cx1 = (x0[s] + lx[s] - 1) / VS_CELL;
            int32_t cy0 = y0[s] / VS_CELL, cy1 = (y0[s] + ly[s] - 1) / VS_CELL;
            int32_t cz0 = z0[s] / VS_CELL, cz1 = (z0[s] + lz[s] - 1) / VS_CELL;
            for (int32_t cz = cz0; cz <= cz1; ++cz)
                for (int32_t cy = cy0; cy <= cy1; ++cy)
                    for (int32_t cx = cx0; cx <= cx1; ++cx) {
                        int64_t cell = ((int64_t)cz * c->cgy + cy) * c->cgx + cx;
                        if (pass == 0) start[cell]++;
                        else items[fillpos[cell]++] = s;
                    }
        }
        if (pass == 1) free(fillpos);
    }
    c->x0 = x0; c->y0 = y0; c->z0 = z0; c->lx = lx; c->ly = ly; c->lz = lz;
    c->ox = ox; c->oy = oy; c->oz = oz; c->peak = peak; c->prof = prof;
    c->cell_start = start;
    return c;
}

void vs_cube_destroy(vs_cube* c) {
    if (!c) return;
    free((void*)c->x0); free((void*)c->y0); free((void*)c->z0);
    free((void*)c->lx); free((void*)c->ly); free((void*)c->lz);
    free((void*)c->ox); free((void*)c->oy); free((void*)c->oz);
    free((void*)c->peak); free((void*)c->prof);
    free((void*)c->cell_start); free((void*)c->cell_items);
    free(c);
}

/* sizes of the variable-length tables, for the device upload */
int64_t vs_cube_nprof(const vs_cube* c) {
    int64_t n = 0;
    for (int32_t s = 0; s < c->nsrc; ++s) {
        int64_t e = (int64_t)c->oz[s] + c->lz[s];
        if (e > n) n = e;
    }
    return n;
}
int64_t vs_cube_ncell(const vs_cube* c) { return (int64_t)c->cgx * c->cgy * c->cgz; }
int64_t vs_cube_nitems(const vs_cube* c) { return c->cell_start[vs_cube_ncell(c)]; }

/* Function-pointer target handed to the oracle for procedural (no dense copy) cubes. */
float vs_cube_voxel(const void* ctx, int64_t x, int64_t y, int64_t z) {
    return vs_voxel((const vs_cube*)ctx, x, y, z);
}

/* dst is a dense [sz][sy][sx] box at offset (bx,by,bz). */
void vs_cube_fill(const vs_cube* c, float* dst, int64_t bx, int64_t by, int64_t bz,
                  int64_t sx, int64_t sy, int64_t sz, int nthreads) {
    if (nthreads < 1) nthreads = 1;
#pragma omp parallel for collapse(2) num_threads(nthreads) schedule(static)
    for (int64_t z = 0; z < sz; ++z)
        for (int64_t y = 0; y < sy; ++y) {
            float* row = dst + (z * sy + y) * sx;
            for (int64_t x = 0; x < sx; ++x) row[x] = vs_voxel(c, bx + x, by + y, bz + z);
        }
}

/* c4 compositing microbenchmark layers: dst is [npix][4]. */
void vs_layer_fill(uint64_t seed, int64_t layer, int64_t pix0, int64_t npix, float* dst, int nthreads) {
    if (nthreads < 1) nthreads = 1;
#pragma omp parallel for num_threads(nthreads) schedule(static)
    for (int64_t i = 0; i < npix; ++i) vs_layer_pixel(seed, (uint64_t)layer, (uint64_t)(pix0 + i), dst + 4 * i);
}
