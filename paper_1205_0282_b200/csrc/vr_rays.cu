/*
 * vr_rays.cu -- the per-ray part of row a4, once per frame pixel.
 *
 * PAPER.md:152 (sec. 2.3.2): "each GPU kernel then starts by calculating its ray's start location,
 * orientation, and intersection with the sub-cube's bounding cube". The ray of a pixel, its clip
 * against the WHOLE volume and its sample schedule (R1, R2, R4, R5, R18) do not depend on the brick,
 * while a pixel's ray crosses several bricks (4.7 on c2, 7 on c3): they are computed here once per
 * pixel of the frame - 18 FP64 divisions and a square root, individually rounded (DESIGN.md
 * "Set-up arithmetic") - and kept in the frame's ray table (vr_internal.cuh), from which the
 * ray-cast kernel starts every (ray, brick) segment with four 16-byte loads and one of 4 bytes. Only the pixels
 * inside the union of the rendering rectangles (VrViewState::bound) are touched.
 */
#include "vr_march.cuh"

#define RAYS_TILE_W 32
#define RAYS_TILE_H 8

__global__ void __launch_bounds__(RAYS_TILE_W * RAYS_TILE_H)
vr_rays_kernel(const VrGrid g, const VrViewState* __restrict__ vs, int W, int H, double step, double2* __restrict__ rays) {
    __shared__ double s_minv[16];
    const int x0 = blockIdx.x * RAYS_TILE_W, y0 = blockIdx.y * RAYS_TILE_H;
    /* tiles outside the union of the rendering rectangles leave after one 16-byte load */
    const int4 bound = *reinterpret_cast<const int4*>(vs->bound);
    if (x0 >= bound.z || x0 + RAYS_TILE_W <= bound.x || y0 >= bound.w || y0 + RAYS_TILE_H <= bound.y) return;
    if (threadIdx.x < 16) s_minv[threadIdx.x] = vs->Minv[threadIdx.x];
    __syncthreads();
    if (vs->singular) return;
    const int i = x0 + (threadIdx.x & (RAYS_TILE_W - 1)), j = y0 + threadIdx.x / RAYS_TILE_W;
    if (i < bound.x || i >= bound.z || j < bound.y || j >= bound.w) return;
    RaySetup r;
    ray_setup(s_minv, W, H, i, j, g, step, r);
    ray_store(rays, (long long)W * H, (long long)j * W + i, step > 0.0, r);
}

cudaError_t vr_launch_rays(const VrGrid& grid, const VrViewState* vs, int W, int H, double step, double2* rays, cudaStream_t st) {
    const dim3 blocks((W + RAYS_TILE_W - 1) / RAYS_TILE_W, (H + RAYS_TILE_H - 1) / RAYS_TILE_H);
    vr_rays_kernel<<<blocks, RAYS_TILE_W * RAYS_TILE_H, 0, st>>>(grid, vs, W, H, step, rays);
    return cudaGetLastError();
}
