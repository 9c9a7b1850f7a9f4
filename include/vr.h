/*
 * vr.h -- C ABI of libvr: the data-parallel hot path of the bricked ray-casting volume
 * renderer of Hassan, Fluke & Barnes, "A Distributed GPU-based Framework for real-time 3D
 * Volume Rendering of Large Astronomical Data Cubes" (arXiv:1205.0282), written from the
 * paper for one NVIDIA B200 (sm_100a).
 *
 * Citations are lines of the paper text with the section they fall in; "R#" are
 * the readings listed in DESIGN.md for points on which the paper is silent.
 *
 * Conventions (all calls)
 *   - Every function returns a vr_status (0 = VR_OK). No exception or C++ type crosses this
 *     boundary. vr_last_error() gives a human-readable message for the last failing call on
 *     a handle (or for a failing vr_volume_create / vr_composite when passed NULL).
 *   - "device" pointers are CUDA device pointers of the current device; "host" pointers are
 *     ordinary process memory. Which one a parameter takes is stated per parameter.
 *   - `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream). Calls
 *     that take a stream are asynchronous on it and never synchronise the host, except where
 *     a HOST output buffer is written (stated per call). Calls without a stream synchronise.
 *   - Ownership: the library owns the brick store and its per-view scratch (rectangles,
 *     visibility order, work list, sub-images). The caller owns every buffer it passes in;
 *     inputs are read (or copied) before the call's work completes on `stream`, outputs are
 *     written by it.
 *   - Geometry: world units are voxels. The volume occupies [0,nx] x [0,ny] x [0,nz]; voxel
 *     (i,j,k) is centred at (i+1/2, j+1/2, k+1/2) (R3). Cube memory layout is [nz][ny][nx]
 *     float32, x fastest, z = spectral axis.
 *   - Blanked voxels: a NaN voxel is blanked (R14). A sample with more than 4e-6 of its tri-linear
 *     weight on NaN voxels is dropped (adds nothing in VR_ALPHA, cannot be the maximum in
 *     VR_MIP); with less, the NaN voxels are left out and the other weights renormalised. The
 *     data range ignores NaN. Infinities are not supported.
 *   - Matrices: column-major float[16], OpenGL clip conventions, clip = proj * view * world,
 *     clip z in [-1,1] (sec. 2.3.2 "the OpenGL projection and transformation
 *     matrices"; R1). Image: [height][width][4] float32 RGBA, row 0 = bottom row, pixel
 *     centres at half-integers.
 *
 *   - Threads and devices: a handle belongs to the CUDA device that was current when it was
 *     created and must be used with that device current. Calls on ONE handle must not
 *     overlap in time (no internal locking); different handles may be used from different
 *     threads. One process drives one GPU (the multi-GPU launch is one process per GPU).
 *   - Environment (experiments only, read by vr_volume_create*): VR_TILE="lx,ly,lz,mx,my,mz"
 *     (log2 micro-tile edge and log2 micro-tiles per macro block and axis; default 2,2,1,0,0,0)
 *     and VR_LAYOUT=1|2 override the brick layout. Results never depend on the layout.
 *
 * There is no CPU fallback: every call needs a CUDA device and fails with VR_ERR_CUDA
 * without one.
 */
#ifndef VR_H
#define VR_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum vr_status {
    VR_OK = 0,
    VR_ERR_INVALID_ARG = 1,   /* bad sizes, NULL pointers, step < 0, singular proj*view ... */
    VR_ERR_OUT_OF_MEMORY = 2, /* a device (or staging) allocation failed */
    VR_ERR_CUDA = 3,          /* a CUDA call or kernel launch failed; see vr_last_error */
    VR_ERR_STATE = 4          /* call order: no transfer function set, no data uploaded ... */
} vr_status;

enum { VR_ALPHA = 0, VR_MIP = 1 };   /* vr_render mode */
#define VR_STEP_AUTO 0.0f            /* vr_render step: the paper's per-ray step (R18) */
enum { VR_HOST = 0, VR_DEVICE = 1 }; /* memory space of a data pointer */
/* Layout of a ghost-padded brick in HBM (north_star: "a tiled linear layout ... whichever ncu
 * shows is faster"). LINEAR: rows of P = brick + 2*ghost cells, x fastest. TILED: 4x4x2-cell
 * micro-tiles of 32 floats = one 128-byte DRAM line each, tiles x fastest, so that the 2x2x2
 * neighbourhoods of consecutive samples of a ray fall into few lines. DEFAULT = TILED (the
 * faster one on every config measured, see DESIGN.md and profiles/). Results do not depend
 * on the layout. */
enum { VR_LAYOUT_DEFAULT = 0, VR_LAYOUT_LINEAR = 1, VR_LAYOUT_TILED = 2,
       /* TILED, with the store's memory mapped brick by brick (CUDA virtual memory management) so that
        * vr_volume_release_store can hand it back; identical to TILED for every other call */
       VR_LAYOUT_TILED_RELEASABLE = 3 };

typedef struct vr_volume vr_volume; /* opaque */

/* Device memory for the library's long-lived buffers (north_star: "PyTorch used only for device
 * memory and streams"). By default libvr takes the brick store, the tables and the per-view scratch from cudaMalloc.
 * After vr_set_allocator(alloc, free, user) every handle created LATER takes them from the caller's allocator instead
 * and returns them to it (the Python binding passes torch's caching allocator: use_torch_allocator()):
 *   alloc(bytes, user) returns a device pointer aligned to 256 bytes, or NULL when out of memory;
 *   free(ptr, user) is called once per pointer, with no work of the library pending on it.
 * A handle keeps the pair it was created with. Both NULL: back to cudaMalloc. Not covered: the 3-D CUDA arrays of
 * the texture arm (cudaMalloc3DArray has no pointer form) and short-lived tables of debug calls. Process-wide, not
 * thread-safe against concurrent vr_volume_create. */
typedef void* (*vr_alloc_fn)(size_t bytes, void* user);
typedef void (*vr_free_fn)(void* ptr, void* user);
int vr_set_allocator(vr_alloc_fn alloc_fn, vr_free_fn free_fn, void* user);

/* Counters of the most recent vr_render on a handle (vr_debug_stats). */
typedef struct vr_stats {
    int64_t samples;        /* tri-linear samples taken (after early termination); valid only
                               if counting was enabled with vr_set_counting, else -1 */
    int64_t rays;           /* (brick, pixel) rays started = sum of launch-rectangle areas */
    int64_t work_items;     /* (brick, 8x4-pixel tile) work items of the ray-cast kernel */
    int64_t subimage_bytes; /* bytes of brick sub-images written by the ray-cast kernel */
    int64_t cells_touched;  /* distinct brick-store cells (float32 voxels) the frame's samples
                               read, and distinct 32-byte sectors (8 consecutive cells) they */
    int64_t sectors_touched;/* fall in; valid only with vr_set_counting(v, 2), else -1 */
    int64_t lines_touched;  /* distinct 128-byte lines (32 consecutive cells) of the brick store
                               they fall in; valid only with vr_set_counting(v, 2), else -1 */
    int32_t nbricks;
    int32_t overflow;       /* 1 if the view needed more sub-image scratch than was reserved
                               (frame is then incomplete; never happens unless the host and
                               device rectangle computations disagree) */
    float ms_setup;         /* per-stage device times of the last render, from CUDA events  */
    float ms_raycast;       /*   recorded on the render's stream; valid only if timing was   */
    float ms_composite;     /*   enabled with vr_set_timing, else -1                         */
    int32_t bricks_culled;  /* bricks the view skipped as transparent (R16); 0 in MIP mode or
                               with culling off */
} vr_stats;

/* ------------------------------------------------------------------------------------------
 * Brick store.
 * PAPER.md:105,113 (sec. 2.1: the cube is split into sub-cubes, each rendered independently at
 * full output resolution), :136 (sec. 2.3.1 partitioning), :146 (data moved to GPU memory).
 * Ghost voxels are not in the paper; R3: each brick carries `ghost` extra voxels per side,
 * edge-replicated at the volume boundary, so that tri-linear sampling is seam-free; ghost = 1
 * is exactly sufficient.
 * ---------------------------------------------------------------------------------------- */

/* Create a volume of nx*ny*nz float32 voxels split into a regular grid of brick^3 cores
 * (ceil(n/brick) per axis, ragged at the high edges). Allocates grid-many padded bricks of
 * (min(brick, max(nx,ny,nz)) + 2*ghost)^3 floats in device memory, zero-filled.
 *   nx,ny,nz > 0; brick >= 2; 0 <= ghost <= 8 (ghost = 0 is allowed: seams are then expected).
 *   out (host): receives the handle. Errors: VR_ERR_INVALID_ARG, VR_ERR_OUT_OF_MEMORY,
 *   VR_ERR_CUDA (no device). On error *out = NULL. */
int vr_volume_create(int nx, int ny, int nz, int brick, int ghost, vr_volume** out);

/* Same, with the brick layout chosen by the caller (VR_LAYOUT_*): vr_volume_create is this
 * call with VR_LAYOUT_DEFAULT. A TILED slot is padded to whole micro-tiles per axis (514^3
 * cells -> 516 x 516 x 514, +0.8 %). Errors as above, plus VR_ERR_INVALID_ARG for an unknown
 * layout. */
int vr_volume_create_layout(int nx, int ny, int nz, int brick, int ghost, int layout, vr_volume** out);

/* Free everything the library allocated for the handle (synchronises the device). NULL ok. */
void vr_volume_destroy(vr_volume* v);

/* Copy a dense box of the cube into the brick store. `src` is a dense [sz][sy][sx] float32
 * array (x fastest) holding the voxels of the box with origin (x0,y0,z0); memspace says
 * whether src is a VR_HOST or VR_DEVICE pointer. Every brick cell (core AND ghost, including
 * the edge-replicated cells outside the volume) whose clamped global voxel index lies in the
 * box is written. A whole-cube upload is (0,0,0,nx,ny,nz); z-slab uploads make the ~100 GB
 * case feasible without a second full copy.
 *   VR_DEVICE: asynchronous on `stream`; src must stay valid until that work completes.
 *   VR_HOST: staged through a bounded device buffer; returns after the copy has completed.
 * Errors: VR_ERR_INVALID_ARG (NULL, box outside the volume, empty box). */
int vr_volume_upload(vr_volume* v, const float* src, int memspace, int x0, int y0, int z0,
                     int sx, int sy, int sz, void* stream);

/* Test-only inverse of vr_volume_upload: reads the CORE cells of the bricks back into a dense
 * [sz][sy][sx] box (dst: VR_HOST or VR_DEVICE). Round trip is bit-exact. VR_HOST synchronises. */
int vr_volume_download(vr_volume* v, float* dst, int memspace, int x0, int y0, int z0,
                       int sx, int sy, int sz, void* stream);

/* Test-only: copy the padded cells of brick b, as a dense [dz][dy][dx] box with
 * d = (core extent + 2*ghost) per axis, to dst (host). dims (host int[3]) receives dx,dy,dz.
 * dst may be NULL to query dims only. Synchronises. */
int vr_debug_brick_data(vr_volume* v, int b, float* dst, int* dims);

/* ------------------------------------------------------------------------------------------
 * Classification (row a6). PAPER.md:45 (sec. 1.2: the transfer function maps a data value to
 * colour and opacity), :172 (final colour mapping with the user's colour map). R7: n-entry
 * straight-alpha RGBA table over [vmin,vmax], values clamped, linear interpolation between
 * entries at x = u*(n-1); the table's alpha is the opacity of one voxel of path length, a
 * sample standing for a path of length w has opacity 1-(1-a)^w.
 *   rgba (host): n*4 floats, copied. 2 <= n <= 1024; vmax > vmin. Synchronises the device
 *   (so that a render in flight is not disturbed). */
int vr_set_transfer_function(vr_volume* v, const float* rgba, int n, float vmin, float vmax);

/* Early ray termination threshold tau (row a7; "... or opacity is achieved").
 * R8: a brick's ray stops, before taking a sample, once the brick-local accumulated opacity
 * is >= tau. Default 0.99; tau > 1 disables early termination. */
int vr_set_early_termination(vr_volume* v, float tau);

/* ------------------------------------------------------------------------------------------
 * Data range. PAPER.md:146 (sec. 2.3.1): "An independent task to
 * determine the local minimum and maximum starts when the data is loaded into the GPU memory";
 * :152 the march may stop at "the maximum pixel value (defined by the global maximum of the
 * data)". Local = per brick, over the brick's ghost-padded cells. The range is computed by one
 * streaming pass over the brick store on the device, lazily, after the last upload: by
 * vr_volume_minmax, or by the first vr_render that wants it (culling on). It gives the caller
 * the data min/max for vr_set_transfer_function, lets MIP rays stop at the global maximum, and
 * lets ALPHA frames skip transparent bricks.
 *   vmin_out, vmax_out (host): range of the whole volume. Runs on `stream`, then waits for it.
 * Errors: VR_ERR_STATE (nothing uploaded), VR_ERR_CUDA. */
int vr_volume_minmax(vr_volume* v, float* vmin_out, float* vmax_out, void* stream);

/* Transparent-brick culling (R16), default ON. In VR_ALPHA mode a brick is skipped for a frame
 * (no rays, no sub-image, not composited) iff every transfer-function entry with index in
 * [max(0, I(min_b) - 1), min(n - 1, I(max_b) + 2)] has alpha == 0, where
 * I(x) = min((int)(sat((x - vmin) * inv_range) * (n - 1)), n - 2) in float32 is the entry a
 * value classifies to; the widening absorbs the rounding of interpolated values. Such a brick
 * contributes exact zeros, so the frame is bit-identical with culling on or off. */
int vr_set_culling(vr_volume* v, int enable);
/* With culling on, VR_ALPHA frames also skip transparent space INSIDE bricks (R19; 4x4x2 layout,
 * ghost >= 1, and only when the transfer function has at least three consecutive entries with
 * alpha == 0 - fewer can never satisfy R16's rule, e.g. the lone zero of a linear ramp). The padded
 * cells of a brick are cut into 8x8x8 macro-cells; macro-cell m is transparent iff R16's rule
 * holds for the (min, max) of cells 8m .. 8m+8 per axis (the macro-cell plus one layer on its
 * high sides) - every voxel a sample based in m can interpolate between. Samples based in a
 * transparent macro-cell are not fetched (a lane leaps to the macro-cell's exit): their opacity is exactly zero, so frames are bit-identical with culling on or
 * off. The per-cell ranges are computed once after an upload (one streaming pass, 8 bytes per 512
 * voxels of extra memory), the transparency bits once per transfer function.
 * VR_MIP frames use the same per-cell ranges where the cube has empty space (at least an eighth
 * of the macro-cells hold nothing but the global minimum, e.g. the zero background of a density
 * cube): a macro-cell whose maximum (plus a rounding margin) cannot raise the ray's running
 * maximum is stepped over; frames stay bit-identical. That decision is taken once per upload by
 * the first VR_MIP frame, which therefore waits once for an 8-byte read-back on its stream. */

/* ------------------------------------------------------------------------------------------
 * One frame (rows a2..a9): per-view set-up (inverse of proj*view, rendering rectangle of each
 * brick = screen bounding box of its 8 projected vertices, Fig. 4 :168),
 * device-side visibility order of the bricks (PAPER.md:53 names depth sorting; R9), per-brick
 * ray casting (sec. 2.3.2: ray start, direction, intersection with the bounding
 * cube, early exit for rays that miss, march to the exit point or until the opacity / the
 * maximum is reached; tri-linear interpolation :69,:150), then sort-last compositing of the
 * brick sub-images in visibility order (sec. 2.3.3: `over` is associative;
 * MIP composites in any order) and, for MIP, the final colour mapping (:172).
 *   view, proj (host): float[16] each, read before the call returns.
 *   width,height > 0; mode VR_ALPHA or VR_MIP.
 *   step > 0: sample spacing along every ray, in voxels (R5). step == VR_STEP_AUTO (0): the
 *   paper's own rule, "a discrete ray-casting with at least one sample for each voxel
 *   intersected": per ray, one sample per unit advance along the ray's major
 *   axis, step = 1 / max(|d_x|,|d_y|,|d_z|) for the unit direction d (R18; 1 .. sqrt(3) voxels).
 *   out_rgba (device): [height][width][4] float32. VR_ALPHA: premultiplied colour and opacity
 *   on a transparent black background. VR_MIP: LUT colour of the ray's maximum with alpha 1,
 *   or (0,0,0,0) if the ray took no sample (R11).
 * Asynchronous on `stream`; all stages run on the device, the host only validates arguments
 * and sizes scratch memory (growing the scratch for a larger view than any seen before
 * allocates, which may synchronise; steady-state frames do not).
 * Errors: VR_ERR_INVALID_ARG (also: proj*view singular), VR_ERR_STATE (no transfer function
 * or nothing uploaded), VR_ERR_OUT_OF_MEMORY, VR_ERR_CUDA. */
int vr_render(vr_volume* v, const float* view, const float* proj, int width, int height,
              float step, int mode, float* out_rgba, void* stream);

/* Size the per-view scratch BEFORE rendering, so that vr_render never allocates and never synchronises the host
 * ("vr_render is asynchronous on the given stream and never syncs the host"): sub-image scratch for
 * the most demanding of the `nviews` given views (+25 %), the ray table and the host entries' device frames for
 * width x height frames. views, projs (host): nviews * 16 floats each, as vr_render takes them. A frame that still
 * needs more (a view not announced here) grows the scratch as before, which synchronises once. A frame whose set-up
 * finds the scratch too small on the DEVICE (host and device rectangle arithmetic would have to disagree by more than
 * the pixel of slack) comes out blank; the next vr_render / vr_render_host* call on the handle returns VR_ERR_STATE. */
int vr_reserve_views(vr_volume* v, const float* views, const float* projs, int nviews, int width, int height);

/* Traversal. VR_SORT_LAST (default) is the path above: every brick
 * renders its own sub-image with BRICK-LOCAL early termination (R8) and the sub-images are
 * composited in visibility order, as the paper's GPUs do.
 * VR_FUSED marches one ray per frame pixel through all the bricks it crosses, front to back,
 * with one accumulator and GLOBAL early termination, and writes the frame directly: no
 * sub-images, no compositing pass. R17: the result is what VR_SORT_LAST gives for a volume
 * held in a single brick (same sample schedule, R5; same voxels, R3), early termination
 * included; with early termination off the two traversals agree to rounding.
 * vr_debug_subimages does not apply to fused frames; transparent bricks (R16) are skipped along
 * the ray, exactly as they are skipped as sub-images. */
#define VR_SORT_LAST 0
#define VR_FUSED 1
int vr_set_traversal(vr_volume* v, int traversal);

/* Sampler of row a5 (north_star: bricks "either as 3D CUDA arrays behind texture objects or as a tiled linear
 * layout with hand-rolled vectorised trilinear interpolation, whichever ncu shows is faster"; the paper's own
 * design is the former, PAPER.md:150 sec. 2.3.2 "built-in tri-linear interpolation", :69).
 * VR_SAMPLER_MANUAL (default): 8 float32 loads from the tiled store and 7 float32 FMA per sample.
 * VR_SAMPLER_TEXTURE: VR_ALPHA frames of the VR_SORT_LAST traversal fetch each sample with one hardware-filtered
 * texture read from a 3-D CUDA array per brick (float32 texels, linear filter, clamp addressing, unnormalised
 * coordinates = R3's voxel-centre convention). The arrays are a SECOND copy of the handle's bricks, allocated
 * by this call (VR_ERR_OUT_OF_MEMORY if they do not fit beside the store - the 103 GB cube - and the sampler
 * is then VR_SAMPLER_MANUAL: arrays of another texel width were freed to make room) and refilled from the store on the device by the first frame after an upload. The sample
 * SET is unchanged (same FP64 set-up); the hardware's 8-bit interpolation weights perturb sample values by up
 * to 2^-9 of the local voxel differences, which keeps VR_ALPHA inside its 2e-3 tolerance but moves early-
 * termination decisions of rays whose opacity passes tau within ~1e-4 of it. The opacity correction 1 - (1 - a)^step
 * multiplies that error by the step and, for steps below one voxel, without bound where the table's opacity nears 1:
 * ALPHA values come from the arrays for 0 < step <= 1 only (larger steps and VR_STEP_AUTO: hand-rolled); with step < 1 a
 * sample whose table opacity exceeds 0.9 is re-evaluated by the hand-rolled sampler, and a ray's (at most two) exit
 * samples are hand-rolled whenever the float32 store exists.
 * VR_MIP frames (1e-5) of the VR_SORT_LAST traversal use the arrays as an EXACT filter: a filtered fetch is within
 * range / 64 (+ 2^-14 of the largest magnitude) of the hand-rolled value for every sample of a brick (the brick's
 * range: row f1), so only samples whose filtered value lies within twice that of the largest one seen on their ray
 * segment can be the segment's maximum; only those are evaluated - by the hand-rolled float32 sampler from the store.
 * The frame is bit-identical to VR_SAMPLER_MANUAL's (a maximum does not depend on the order of its operands); it
 * needs both copies (not a released store) and is not combined with stepping over empty macro-cells (R19: where
 * that pays, it is used instead). Fused MIP frames
 * and counting mode 2 always use the hand-rolled path, and so do (i) bricks that hold blanked (NaN) voxels -
 * the filter cannot apply R14's rule - and (ii) frames whose transfer function has a step: two neighbouring entries
 * further apart than 1.1/n in a channel - anything steeper than a ramp over the table's whole range (a threshold, a toe,
 * a ramp over half the range). The filter's value error is about one table entry on unit-sigma noise, so the frame's
 * error grows with the table's slope: 1.4e-3 to 1.65e-3 at slope 1 (the ramp), 2.7e-3 at 1.5, 3.3e-3 at 2.5, 8e-2 on
 * a threshold table (measured). (iii) For the same reason the data must be smooth enough against the table: with R = the
 * mean range of the 8x8x8 macro-cells over the table's range (0.46-0.48 on the benchmark cubes), VR_ALPHA values come
 * from the arrays only while 3.5e-3 x R x (table slope) <= 1.9e-3 (vr_debug_tex_alpha_guard); otherwise the frames use
 * the hand-rolled sampler (VR_ERR_STATE on a released store). Needs ghost >= 1 (the macro-cell table).
 * VR_SAMPLER_TEXTURE_HALF: the same arm with arrays of float16 texels - float16 COPIES of the float32 voxels, made for
 * sampling only (the store, the range tables, blanked bricks and every other path stay float32): half the memory and
 * about three quarters of the fetched bytes. Rounding a voxel to float16 (to nearest) moves it by at most 2^-11 of its
 * magnitude and the unit filters such texels at float16 precision (2^-10 in all) - for data of a few sigma half of what
 * the filter's 8-bit weights already move a sample (2^-9 of the local voxel differences) - so VR_ALPHA frames stay inside 2e-3 (measured against the oracle: the same error as with
 * float32 texels to two digits, R22). Guard: while the largest magnitude in the volume / 1024 exceeds 1.5e-3 of
 * the transfer function's range, VR_ALPHA frames use the hand-rolled sampler instead (VR_ERR_STATE on a released store):
 * float32 texels are for such data. For VR_MIP the arrays are the exact filter described above, the bound carrying the
 * rounding (range / 64 + 2^-9 of the brick's largest magnitude + 2^-23 for float16's subnormal grid); bricks holding a magnitude above 60000 (float16
 * ends at 65504) keep the hand-rolled loop: VR_MIP frames stay bit-identical to VR_SAMPLER_MANUAL's. These arrays fit
 * beside the 103 GB cube (105 GB store + 53 GB).
 * VR_SAMPLER_TEXTURE_BYTE: the same filter with 8-bit texels, q = round(255 (v - min) / (max - min)) with the brick's own
 * range (row f1's table, computed first): a quarter of the float32 arrays' memory and the fewest fetched bytes; the
 * bound grows by half a byte step (range / 64 + range / 500 + 2^-12 of the largest magnitude). VR_MIP frames
 * bit-identical to VR_SAMPLER_MANUAL's as well; VR_ALPHA frames use the hand-rolled sampler (8 bits would not keep 2e-3).
 * Switching to VR_SAMPLER_MANUAL, or between texel widths, frees the arrays (synchronises the device).
 * Needs the default (tiled) layout. */
#define VR_SAMPLER_MANUAL 0
#define VR_SAMPLER_TEXTURE 1
#define VR_SAMPLER_TEXTURE_HALF 2
#define VR_SAMPLER_TEXTURE_BYTE 3
int vr_set_sampler(vr_volume* v, int sampler);

/* The texture arm for cubes whose second copy does not fit beside the store (the 103 GB cube).
 * On a handle created with VR_LAYOUT_TILED_RELEASABLE and filled: computes the range tables (rows f1, R19) if they are
 * stale, then, brick by brick, creates the brick's 3-D array, fills it from the float32 store and gives the brick's
 * float32 cells back to the device (peak memory: the store plus one array). Bricks that hold blanked (NaN) voxels keep
 * their float32 cells, because R14 needs them. The arrays take the texel width of the sampler in force (float16 after
 * vr_set_sampler(v, VR_SAMPLER_TEXTURE_HALF), else float32). Afterwards the handle renders VR_ALPHA frames (both traversals) through the
 * texture arm only: vr_volume_upload / download, VR_MIP frames, counting mode 2, transfer functions with a step and
 * sample steps outside [0.9, 1] voxels (see vr_set_sampler: smaller steps need the float32 store for their guard)
 * return VR_ERR_STATE. Irreversible; synchronises. freed_bytes_out (host, may be NULL): device memory given back.
 * Errors: VR_ERR_STATE (not a releasable handle, nothing uploaded, already released), VR_ERR_OUT_OF_MEMORY, VR_ERR_CUDA. */
int vr_volume_release_store(vr_volume* v, int64_t* freed_bytes_out, void* stream);

/* Same frame, delivered to HOST memory: renders into a library-owned device frame, copies it
 * to out_rgba_host ([height][width][4] float32; pinned memory makes the copy asynchronous
 * with respect to other streams) and waits for the copy. This is the end-to-end entry. */
int vr_render_host(vr_volume* v, const float* view, const float* proj, int width, int height,
                   float step, int mode, float* out_rgba_host, void* stream);

/* The same end-to-end frame, PIPELINED: the call returns once the frame's kernels and its
 * device->host copy are queued, and the copy of frame i (on a library-owned copy stream, out
 * of one of two library-owned device frames) overlaps the rendering of frame i+1 on `stream`.
 * This is how a frame server uses the renderer (the server renders while the
 * previous frame travels to the viewer).
 *   out_rgba_host (host, should be pinned): [height][width][4] float32; its contents are
 *   defined only after vr_render_host_wait returns. The caller must not reuse the buffer for
 *   another frame before that (use one buffer per frame in flight; two frames are in flight).
 * vr_render_host_wait blocks until every frame queued by vr_render_host_async on this handle
 * has arrived in host memory. Errors as vr_render; the wait returns VR_ERR_CUDA if a queued
 * copy failed. */
int vr_render_host_async(vr_volume* v, const float* view, const float* proj, int width,
                         int height, float step, int mode, float* out_rgba_host, void* stream);
int vr_render_host_wait(vr_volume* v);

/* ------------------------------------------------------------------------------------------
 * Stand-alone sort-last compositing (row a9; the 64-layer microbenchmark). PAPER.md:114
 * (compositing is the bottleneck of distributed image-order rendering), :170-174.
 *   layers (host array of n DEVICE pointers): layer l is a premultiplied RGBA float32
 *   sub-image covering rects[l], stored [y1-y0][x1-x0][4].
 *   rects (host): n * (x0,y0,x1,y1), half-open, inside the width x height viewport.
 *   order (host): n layer indices, front to back.
 *   out (device): [height][width][4]; pixels no layer covers become (0,0,0,0).
 * Front-to-back `over`: C += (1-A)*C_l, A += (1-A)*A_l, float32 (R15). Asynchronous on
 * `stream` after copying the small tables (n <= 4096). */
int vr_composite(const float* const* layers, const int* rects, const int* order, int n,
                 int width, int height, float* out, void* stream);

/* The same operation for callers that must not allocate (code under CUDA graph capture, tight serving loops,
 * harnesses that forbid cudaMalloc): vr_composite takes its two small device tables from cudaMallocAsync; this
 * entry keeps them in a fixed __device__ array inside the library (11 KB, held by every GPU that loads libvr until
 * the process exits) and calls no cudaMalloc / cudaFree / allocating routine, on the host side either.
 *   Arguments, layouts and result exactly as vr_composite (same kernel: the frames are bit-identical), except
 *   n <= VR_COMPOSITE_STATIC_MAX_LAYERS: more layers -> VR_ERR_INVALID_ARG, nothing launched.
 *   All calls share the one array per device, and it keeps the last call's tables (a call rewrites the entries it
 *   reads; nothing has to be cleared). Calls on one stream are ordered by the stream; calls that OVERLAP on the GPU
 *   (different streams without a dependency) race on the tables: serialise them.
 * Errors: VR_ERR_INVALID_ARG (NULL, n, rectangles, order not a permutation), VR_ERR_CUDA. */
#define VR_COMPOSITE_STATIC_MAX_LAYERS 256
int vr_composite_static(const float* const* layers, const int* rects, const int* order, int n,
                        int width, int height, float* out, void* stream);

/* ------------------------------------------------------------------------------------------
 * Multi-GPU sort-last (PAPER.md:136-138 data partitioning,
 * :170-174 two-stage compositing, :178-184 direct send of rectangle-packed partial frames).
 * One process per GPU; each holds a PART: a box of bricks of the global brick grid. A part
 * handle behaves like a volume in every call above, in GLOBAL voxel coordinates and with the
 * global brick numbering, but stores, ranges, culls and renders only its own bricks: rays,
 * sample positions, the owner rule and the visibility order are those of the whole volume, so
 * the sub-images of a part's bricks are bit-identical to the ones a single handle renders.
 * libvr moves no data between GPUs: the exchange is the caller's (paper_1205_0282_b200.sortlast
 * uses torch.distributed), the partition, the part order, the rectangles and the kernels on both sides of it are these.
 *
 * vr_volume_create_part: b0, b1 (host, int[3]): the part holds bricks b0 <= (bx,by,bz) < b1
 *   (brick (bx,by,bz) = voxels [bx*brick, min((bx+1)*brick, n)) per axis). Memory: the box's
 *   bricks only. vr_volume_upload takes boxes anywhere in the volume and keeps what falls into
 *   the padded extent of the part's bricks: upload the part's voxels plus `ghost` layers of its
 *   neighbours' (R3; a ghost layer left out reads as zeros). vr_volume_download and
 *   vr_debug_brick_data accept the part's own bricks only; vr_volume_minmax gives the range of
 *   the part's voxels (ghost layers included) - reduce it over the parts for the global range;
 *   table entries of bricks held elsewhere are (+inf, -inf).
 * vr_kd_partition: the data partition (sec. 2.3.1: k-d trees; host arithmetic, no handle, no device).
 *   The brick grid is cut across its longest axis (in voxels, ties to the lower axis) at the brick face nearest to
 *   the wanted share (ties to even), at least one brick per side, until there are nparts boxes: nparts = 2^k gives
 *   one balanced tree, other counts a chain of balanced trees, one per set bit of nparts from the largest down,
 *   whose roots share the box in proportion to their leaf counts (6 = 4 + 2).
 *   boxes_out (host, int[nparts*6]): part r holds bricks (b0x,b0y,b0z) <= b < (b1x,b1y,b1z), low side first.
 *   tree_out (host, int[(2*nparts-1)*4]): node 0 = root, pre-order; an inner node is (axis, cut in bricks, low child,
 *   high child), a leaf (-1, part, 0, 0). Errors: VR_ERR_INVALID_ARG (more parts than the grid can be cut into).
 * vr_part_order: the parts front to back for a view (`over` needs a visibility order): at every node
 *   the side of the cut plane that holds the eye first (orthographic: the side the view direction leaves first);
 *   the eye is R9's homogeneous eye from the library's own inverse of proj*view. order_out (host, int[nparts]).
 * vr_render_part: one frame of the part's bricks only, the full frame:
 *   VR_ALPHA  [height][width][4]: premultiplied RGBA of the part's sub-images composited in visibility order
 *             (what vr_render gives on a part handle);
 *   VR_MIP    [height][width]: ONE float per pixel as in the paper (a 1024^2 sub-frame is 4 MB) - the
 *             raw maximum over the part's samples, -inf for a ray that takes no sample in the part (needs
 *             VR_SORT_LAST, else VR_ERR_STATE);
 *   rect_out (host, int[4], may be NULL): (x0,y0,x1,y1), half-open: a rectangle that contains
 *   every non-blank pixel of the partial frame (union of the bricks' rendering rectangles with
 *   a pixel of slack; PAPER.md:184 packs messages by it); all zero if nothing is on screen.
 * vr_render_part_pieces: the same partial frame, composited (stage 1) straight into `npieces`
 *   rectangle-packed pieces instead of a full frame - what a rank sends: piece q covers piece_rects[q] =
 *   (x0,y0,x1,y1) inside the frame (host int[npieces*4]) and is stored [y1-y0][x1-x0][4] (VR_ALPHA) or [y1-y0][x1-x0]
 *   (VR_MIP) at pieces[q] (host array of npieces DEVICE pointers). Only those pixels are written: nothing else of the
 *   frame is touched or cleared. Needs VR_SORT_LAST.
 * vr_part_rect: the same rectangle from the geometry alone (host arithmetic, no handle, no
 *   device), so that every process can size the pieces it will receive without a message.
 * vr_composite_parts: merges partial frames. parts/rects/order/n/out as vr_composite (piece l
 *   covers rects[l]); order = the parts front to back (any order for VR_MIP). VR_ALPHA: pieces
 *   stored [y1-y0][x1-x0][4], front-to-back `over` (identical to vr_composite). VR_MIP: scalar
 *   pieces stored [y1-y0][x1-x0] (-inf = no sample): their maximum, then the colour mapping with v's
 *   transfer function, (0,0,0,0) where no piece holds a sample.
 *   `over` is associative: merging the parts' frames in part order equals
 *   compositing all sub-images in brick order up to float32 rounding, provided the part order
 *   is a visibility order of the boxes (sortlast.part_order: the k-d tree, near side first). */
int vr_volume_create_part(int nx, int ny, int nz, int brick, int ghost, const int* b0,
                          const int* b1, vr_volume** out);
int vr_render_part(vr_volume* v, const float* view, const float* proj, int width, int height,
                   float step, int mode, float* out_part, int* rect_out, void* stream);
int vr_render_part_pieces(vr_volume* v, const float* view, const float* proj, int width, int height,
                          float step, int mode, const int* piece_rects, float* const* pieces, int npieces,
                          void* stream);
int vr_part_rect(int nx, int ny, int nz, int brick, const int* b0, const int* b1,
                 const float* view, const float* proj, int width, int height, int* rect_out);
int vr_kd_partition(int nx, int ny, int nz, int brick, int nparts, int* boxes_out, int* tree_out);
int vr_part_order(const int* tree, int nparts, int brick, const float* view, const float* proj,
                  int* order_out);
int vr_composite_parts(vr_volume* v, int mode, const float* const* parts, const int* rects,
                       const int* order, int n, int width, int height, float* out, void* stream);

/* ------------------------------------------------------------------------------------------
 * Debug / test exports. All synchronise and write HOST memory.
 * ---------------------------------------------------------------------------------------- */

int vr_num_bricks(const vr_volume* v);

/* Front-to-back permutation of the bricks for this view, as computed by the device set-up
 * kernel (R9). order_out: host int[nbricks]. Brick index b = (bz*gy + by)*gx + bx. */
int vr_debug_brick_order(vr_volume* v, const float* view, const float* proj, int* order_out);

/* Rendering rectangle (x0,y0,x1,y1), half-open and clipped to the viewport, of every brick,
 * as computed by the device set-up kernel. rects_out: host int[nbricks*4]. */
int vr_debug_rects(vr_volume* v, const float* view, const float* proj, int width, int height,
                   int* rects_out);

/* Per listed pixel (pixels: host int[npix*2] = (i,j) pairs), the bricks whose core box
 * overlaps the ray's clipped segment with positive length, by increasing entry distance
 * (R10). counts: host int[npix]; lists: host int[npix*maxlen] (entries beyond the count are
 * -1); grazing: host uint8[npix] or NULL, 1 where some hit/miss decision had a margin below
 * 1e-9 voxel (such rays are excluded from exact comparison). */
int vr_debug_ray_bricks(vr_volume* v, const float* view, const float* proj, int width,
                        int height, const int* pixels, int npix, int* counts, int* lists,
                        int maxlen, uint8_t* grazing);

/* Per listed pixel, the sub-image value each brick produced in the most recent vr_render on
 * this handle with the same width/height (test access to row a8). sub_out: host
 * float[npix*nbricks*4]: VR_ALPHA premultiplied RGBA; VR_MIP (max, 0, 0, 0) with max = -inf
 * for "no sample". Bricks whose rectangle does not contain the pixel give zeros / -inf. */
/* Macro-cell transparency flags of brick b under the current transfer function (R19).
 * dims (host): 3 ints, macro-cells per axis of a brick slot; flags_out (host, may be NULL to ask
 * for dims only): dims[0]*dims[1]*dims[2] bytes, x fastest, 1 = transparent. */
int vr_debug_cell_flags(vr_volume* v, int b, unsigned char* flags_out, int* dims);

/* mm_out (host): nbricks * 2 floats, (min, max) per brick over its ghost-padded cells. */
int vr_debug_brick_minmax(vr_volume* v, float* mm_out);

/* The texture arm's data guard for VR_ALPHA values (R20 vii; test / measurement export): the mean range
 * (max - min) of the handle's 8x8x8 macro-cells, the table's largest difference between neighbouring entries in units of
 * 1/n, and whether 3.5e-3 x (mean range / table range) x slope <= 1.9e-3, i.e. whether VR_ALPHA frames may take their
 * values from the arrays (else they use the hand-rolled sampler; VR_ERR_STATE on a released store). Outputs: host.
 * Synchronises. Errors: VR_ERR_STATE (no data or no transfer function). */
int vr_debug_tex_alpha_guard(vr_volume* v, float* mean_cell_range_out, float* table_slope_out, int* ok_out);

/* R23's constant, measured (test / measurement export): with a texture sampler in force, the largest
 * |filtered fetch - exact tri-linear value| over n hashed sample positions inside brick b (the exact value in double
 * from the float32 store; 8-bit fetches decoded with the brick's range), and the brick's range (max - min, row f1).
 * The exact MIP filter relies on max_err <= range / 64 (+ the magnitude terms of vr_set_sampler's text).
 * max_err_out, range_out: host. Synchronises. Errors: VR_ERR_STATE (manual sampler, released store, no data). */
int vr_debug_tex_error(vr_volume* v, int b, int64_t n, unsigned seed, float* max_err_out, float* range_out);

int vr_debug_subimages(vr_volume* v, const int* pixels, int npix, float* sub_out);

/* Counting in the ray-cast kernel (an instrumented variant of the same kernel: slower, never
 * used for timed runs): 0 = off, 1 = count samples, 2 = count samples and keep a bitmap of
 * the brick-store cells read (1 bit per cell of extra device memory), from which
 * vr_debug_stats reports the frame's distinct cells and 32-byte sectors. */
int vr_set_counting(vr_volume* v, int enable);

/* Enable (1) / disable (0) CUDA-event timing of the three stages on the render's stream. */
int vr_set_timing(vr_volume* v, int enable);

/* Counters (and stage times) of the most recent vr_render. Synchronises. */
int vr_debug_stats(vr_volume* v, vr_stats* out);

/* Device times (ms) of set-up, ray casting and compositing of the last `nframes` frames
 * rendered since vr_set_timing(v, 1), oldest first: ms_out (host) float[nframes*3],
 * 1 <= nframes <= 64. Lets a caller time frames back to back without synchronising between
 * them and read every frame's stage times afterwards. Synchronises. */
int vr_debug_stage_times(vr_volume* v, int nframes, float* ms_out);

/* DRAM fetch-granularity probe (no handle). Measures what
 * bounds row a5 on sparsely sampled cubes: the cost of a 4-byte load that misses L2. ctas x 256
 * threads each issue loads_per_thread (a multiple of 8 and of `group`) independent loads at hashed
 * 32-byte-aligned offsets of buf (device, `bytes` long, far larger than L2, any finite contents);
 * the loads of one group of `group` consecutive loads fall into `group` distinct 128-byte lines of
 * one aligned span_bytes block (a power of two >= 128; group <= span_bytes / 128).
 *   flavour: 0 ld.global, 1 ld.global.nc (= __ldg, the ray-cast kernel's load), 2 .cg, 3 .cs, 4 .cv,
 *            5 .nc.L1::no_allocate, 6 .nc.L1::no_allocate.L2::64B, 7 .nc.L2::128B, 8 .nc.L2::256B,
 *            9 .nc.v4.f32 (16 bytes), 10 .nc.L2::64B;
 *            through texture objects: 11 tex1Dfetch<float> and 12 tex1Dfetch<float4> over the head of buf as linear
 *            memory (as far as the device's 1-D linear texture limit reaches); 13 tex3D<float4> point fetches and
 *            14 tex3D<float> linear-filtered fetches (the texture arm's) at hashed positions of a 3-D CUDA array of
 *            1024 x 1024 x (bytes / texel / 2^20, at most 2048) texels which the call allocates and frees (buf may be
 *            NULL; span_bytes / group are ignored)
 *   l2_fetch_granularity: 0 = leave, or 32 / 64 / 128 = cudaLimitMaxL2FetchGranularity (stays set).
 *   ms_out (host): device time of one launch (CUDA events on `stream`, after one warm-up launch);
 *   loads_out (host): loads that launch issued. DRAM bytes per load come from ncu's
 *   dram__bytes_read.sum of the same launch. Synchronises. */
int vr_debug_probe_dram(const void* buf, uint64_t bytes, int flavour, int span_bytes, int group,
                        int loads_per_thread, int ctas, int l2_fetch_granularity, float* ms_out,
                        uint64_t* loads_out, void* stream);

/* Which kernel vr_volume_upload uses for the default (4x4x2) layout, process-wide: 1 (default) = source boxes loaded by the
 * TMA unit (cp.async.bulk.tensor; needs sx % 4 == 0 and a 16-byte aligned source, else falls back to 0), 0 = cp.async
 * staging. Both give the same store, bit for bit; the switch exists to measure one against the other
 * (round 2, c3: 5.86 TB/s against 5.23 TB/s). */
int vr_debug_set_upload_path(int path);

/* Number of kernel launches the library has issued on this handle since creation. */
int64_t vr_launch_count(const vr_volume* v);

/* Message for the last error on the handle (or the last handle-less error if v is NULL).
 * Never NULL; valid until the next call on the same handle. */
const char* vr_last_error(const vr_volume* v);

#ifdef __cplusplus
}
#endif

#endif /* VR_H */
