/* include/vr.h — C ABI of libvr: ray-casting volume rendering of float32 spectral cubes on one
 * B200 (sm_100a).  The boundary of BASELINE.json `north_star` item (1): "a small C-ABI library
 * (upload_cube, set_view, set_transfer_function, render_mip, render_ea, composite_bricks) whose
 * calls follow the paper's statement of the problem" - data file + orientation + colour map +
 * output size -> image (section 2 "colour map"; lines 37-45 section 3 "a static
 * image of the current data file with the same orientation information but with a different
 * output size (defined by the user)"; line 13 abstract "using the ray-casting algorithm";
 * line 57 footnote 4, float32 voxels).  SURVEY.md section 8(b) lists the calls; DESIGN.md states
 * every reading (O-1 ... O-12) the arithmetic follows.
 *
 * Conventions
 *  - Every function returns an int status: 0 = VR_OK, negative = error.  No exceptions, no
 *    aborts.  `vr_last_error(ctx)` returns the text of the last error of that context.
 *  - "d_" arguments are DEVICE pointers, "h_" arguments are HOST pointers.  Large buffers (cube,
 *    meta, frames, partial images) are CALLER-OWNED device memory (e.g. torch tensors); the
 *    library never allocates O(cube) or O(frame) memory.  It owns only small device scratch:
 *    the transfer-function tables (8 KiB), counters, the source lists of the generator, the
 *    descriptors of partial images (<= ~100 B per brick) and, while vr_upload_cube streams a HOST
 *    source, two staging slabs of about 128 MiB each (freed before the call returns).
 *  - `stream` is a cudaStream_t passed as void* (torch.cuda.current_stream().cuda_stream); work
 *    is enqueued on it and no call synchronises the device unless stated.  Outputs are valid
 *    after the caller synchronises the stream.
 *  - One context per host thread; a context is bound to one device.
 *  - Voxel (i,j,k) = (RA, Dec, frequency) sits at integer position (i,j,k); the rendered domain
 *    is the closed box [0,nx-1] x [0,ny-1] x [0,nz-1] (O-1).  Linear cubes are x-fastest.
 *  - Dimensions need not be multiples of the brick size (1721 x 1721 x 1025);
 *    edge bricks are partial.  Voxels must be finite.
 */
#ifndef VR_H
#define VR_H
#include <stddef.h>
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct vr_ctx vr_ctx;

enum {
    VR_OK = 0,
    VR_ERR_INVALID_ARG = -1, /* null pointer, non-positive size, vmax <= vmin, step <= 0, singular matrix */
    VR_ERR_BUFFER = -2,      /* a caller buffer is too small */
    VR_ERR_CUDA = -3,        /* a CUDA call failed; text kept in vr_last_error */
    VR_ERR_STATE = -4,       /* render before cube / view / transfer function were set */
    VR_ERR_UNSUPPORTED = -5
};
enum { VR_MODE_MIP = 0, VR_MODE_EA = 1 };

/* ---- lifetime ------------------------------------------------------------------------------ */
int vr_create(vr_ctx** out, int device);
int vr_destroy(vr_ctx* ctx);
const char* vr_last_error(const vr_ctx* ctx);
const char* vr_status_string(int status);

/* ---- S0: cube residency (BASELINE.json north_star (2),(4)) -------------- */
/* Bytes the caller must allocate for the brick-major cube (bricks of bx*by*bz voxels stored with
 * a one-sided +1 halo, x pitch padded to a multiple of 4 floats) and for its metadata (per-brick
 * and per-8^3-cell (min,max) over the halo-inclusive voxel set, plus activity bits: one per brick,
 * per macro-cell and per voxel, and a scratch bit per voxel for their classification: 2/32 of the cube). */
int vr_cube_layout(int nx, int ny, int nz, int bx, int by, int bz, size_t* cube_bytes,
                   size_t* meta_bytes);

/* The same for the micro-block layout (VR_OPT_LAYOUT 1, the default) with a stored voxel type (VR_OPT_VOXEL_TYPE:
 * 0 = float32, 1 = float16, half the bytes) and a window of resident bricks (end_brick < 0: all bricks). */
int vr_cube_layout_typed(int nx, int ny, int nz, int bx, int by, int bz, int voxel_type, int first_brick, int end_brick,
                         size_t* cube_bytes, size_t* meta_bytes);

/* Bytes at the START of d_meta that depend on the cube alone ((min,max) per brick and per macro-cell); the rest is
 * classification against the current transfer function, which the library recomputes on the device when a render
 * needs it.  A caller that keeps (a window of) a cube outside HBM and brings it back later (PAPER.md
 * line 19: cubes "larger than a single machine memory limit"; paper_1012_2909_b200/outofcore.py) saves and restores the cube
 * bytes and these leading meta bytes, then calls vr_attach_cube. */
int vr_meta_static_bytes(int nx, int ny, int nz, int bx, int by, int bz, int voxel_type, int first_brick, int end_brick,
                         size_t* static_bytes);

/* Rebrick a linear x-fastest float32 cube (host if src_is_device == 0, else device) into d_cube
 * and compute d_meta.  Host sources are streamed slab by slab (whole planes) through two library
 * staging slabs, the copy of one overlapping the rebricking of the other; the call synchronises `stream`.
 * Non-finite voxels (NaN, inf) are counted while rebricking: VR_ERR_INVALID_ARG, and no cube is set. */
int vr_upload_cube(vr_ctx* ctx, const float* src, int src_is_device, int nx, int ny, int nz,
                   int bx, int by, int bz, void* d_cube, void* d_meta, void* stream);

/* Device-side generator of the synthetic cubes (north_star (4); recipe SURVEY.md 8(d)):
 * value(x,y,z) = N(0,1) noise from a counter-based hash of (seed, x + nx (y + ny z))
 *              + continuum * z / (nz - 1) + sum of the sources whose integer box holds (x,y,z),
 * zero inside the zero boxes; written brick-major in place, then d_meta is computed. */
typedef struct {
    const double* h_sources; /* n_sources x 16 doubles: x0 y0 z0 amp sigma_a sigma_b sigma_z
                                cos sin gradient xlo xhi ylo yhi zlo zhi (boxes inclusive) */
    int n_sources;
    const int* h_zero_boxes; /* n_zero_boxes x 6 ints: xlo xhi ylo yhi zlo zhi (inclusive) */
    int n_zero_boxes;
    double continuum;
} vr_gen_params;
int vr_generate_cube(vr_ctx* ctx, const vr_gen_params* params, uint64_t seed, int nx, int ny,
                     int nz, int bx, int by, int bz, void* d_cube, void* d_meta, void* stream);

/* Attach an already resident brick-major cube + meta (e.g. after a context was re-created). */
int vr_attach_cube(vr_ctx* ctx, int nx, int ny, int nz, int bx, int by, int bz, const void* d_cube,
                   void* d_meta);

/* Copy brick `brick_id` (= bx_i + gx (by_i + gy bz_i)) without halo, clipped to the cube, x
 * fastest, into d_dst (device, >= ex*ey*ez floats).  Used to hand cube bytes to a checker. */
int vr_download_brick(vr_ctx* ctx, int brick_id, float* d_dst, void* stream);

/* ---- S1: per-view / per-TF state (O-2, O-6, O-9) ------------------------ */
/* mvp: row-major 4x4, clip = M (x,y,z,1)^T in voxel coordinates, GL clip space.  width/height:
 * the image this matrix maps to.  step_voxels: sampling step Delta.  Resets the viewport to
 * (0, 0, pitch = width). */
int vr_set_view(vr_ctx* ctx, const float mvp[16], int width, int height, float step_voxels);
/* Place the width x height image at pixel (x0, y0) of a larger frame whose rows are pitch_px
 * pixels apart (5 x 5 panels of 1920 x 1080 in one 9600 x 5400 frame). */
int vr_set_viewport(vr_ctx* ctx, int x0, int y0, size_t pitch_px);
/* rgba: 256 entries (r,g,b,a) in [0,1], a = opacity per unit voxel length; values map linearly
 * from [vmin, vmax] onto entries 0..255, clamped, linear between entries (O-6). */
int vr_set_transfer_function(vr_ctx* ctx, const float rgba[256 * 4], float vmin, float vmax);

/* ---- S2-S4: the ray marcher, whole frame, one accumulator per ray (O-8 GLOBAL) ------------- */
/* MIP (O-5): d_out_scalar[(y0+j)*pitch + x0+i] = max over taken samples, or miss_value.  If
 * d_out_rgba_or_null != NULL it receives the raw transfer function evaluated at that maximum
 * ((0,0,0,0) for a miss). */
int vr_render_mip(vr_ctx* ctx, float* d_out_scalar, float* d_out_rgba_or_null, float miss_value,
                  void* stream);
/* Emission-absorption (O-7): front-to-back, early ray termination once alpha >= ert_tau
 * (> 1 disables), result = premultiplied colour over bg, 4 floats per pixel. */
int vr_render_ea(vr_ctx* ctx, float* d_out_rgba, const float bg[4], float ert_tau, void* stream);

/* ---- S5: sort-last path (north_star: "per-brick partial images are then composited sort-last
 *      in visibility order"; O-8 SORT-LAST, O-9) ------------------------------------------- */
typedef struct {
    int brick;        /* brick id */
    int x0, y0, w, h; /* screen rectangle in view pixels (inside [0,width) x [0,height)) */
    void* d_data;     /* device: w*h pixels, row pitch `pitch_px`; EA float4, MIP float */
    size_t pitch_px;
} vr_partial;

/* Front-to-back order of the bricks that can contribute under the current view (inside the
 * frustum; for VR_MODE_EA also active against the transfer function, O-10).  h_order_or_null
 * receives *n_active brick ids (room for all bricks). */
int vr_sort_bricks(vr_ctx* ctx, int mode, int* h_order_or_null, int* n_active);
/* Screen rectangles of n bricks and a packing of their partial images into one arena: fills
 * h_partials[i] (brick, rect, pitch; d_data = byte OFFSET into the arena) and *arena_bytes. */
int vr_partial_layout(vr_ctx* ctx, int mode, const int* h_brick_ids, int n, vr_partial* h_partials,
                      size_t* arena_bytes);
/* Render the partial image of each listed brick: premultiplied (C_b, A_b) with ERT local to the
 * brick (EA) or the brick's maximum, -inf where no sample falls in it (MIP). */
int vr_render_bricks(vr_ctx* ctx, int mode, const vr_partial* h_partials, int n, float ert_tau,
                     void* stream);
/* Fold n partial images in the given order (h_partials[0] in front): over-operator then bg (EA),
 * max then miss value bg[0] (MIP), into the viewport of d_out. */
int vr_composite_bricks(vr_ctx* ctx, int mode, const vr_partial* h_partials, int n, float* d_out,
                        const float bg[4], void* stream);
/* The same fold for callers that must not allocate (code under CUDA graph capture, tight serving loops, harnesses that
 * forbid cudaMalloc): vr_composite_bricks keeps the device copy of the descriptors in a buffer it cudaMallocs on its first
 * call and whenever n grows; this variant keeps it in a static __device__ array of the library instead (224 KiB, held by
 * every GPU that loads libvr until the process exits) and calls no cudaMalloc, cudaFree or other allocating routine, on
 * the device or on the host.  Arguments, result (bit for bit) and error behaviour as vr_composite_bricks, plus: n above
 * VR_STATIC_MAX_PARTIALS is refused with VR_ERR_BUFFER (vr_last_error says so) and nothing is launched.  All calls on a
 * device share the one array: a call rewrites entries [0, n) before its kernel reads them and reads no others, so nothing
 * needs clearing between calls; calls that overlap on the GPU (different streams without an event between them, or
 * different contexts of one device) race on it - order them. */
#define VR_STATIC_MAX_PARTIALS 4096
int vr_composite_bricks_static(vr_ctx* ctx, int mode, const vr_partial* h_partials, int n, float* d_out,
                               const float bg[4], void* stream);

/* The four calls above for the current view in one: the resident bricks that can contribute are sorted front to back
 * (O-9), their partial images are packed into d_arena (device, 256-byte aligned, arena_bytes; *needed_bytes receives
 * what this view needs: VR_ERR_BUFFER and nothing launched if that is more), rendered (S2-S4) and folded into the
 * viewport of d_out (S5).  Same kernels and the same frame as the four calls; the descriptors travel once, through a
 * pinned staging ring of the library, so a frame (or one panel of a tiled frame) costs one call and no host allocation.
 * Up to 32 calls may be in flight on DIFFERENT streams (e.g. the panels of a tiled frame, each with its own arena
 * and viewport): each call has its own descriptor slot; the classification a new table needs is enqueued by the
 * first call that sees it, so order that call before the others (one event). */
int vr_render_sortlast(vr_ctx* ctx, int mode, float ert_tau, void* d_arena, size_t arena_bytes, size_t* needed_bytes,
                       float* d_out, const float bg[4], void* stream);

/* ---- sharding the bricks over several GPUs (PAPER.md line 13 abstract
 *      and line 19 section 1: "distributed GPUs", sub-volumes rendered where they reside and
 *      composited) ----------------------------------------------------------------------------- */
/* Make bricks [first_brick, end_brick) (global ids, x fastest) the only resident ones of this
 * context: read by the next vr_generate_cube / vr_upload_cube / vr_attach_cube, whose d_cube and
 * d_meta then hold just these bricks (sizes: vr_window_layout).  All calls keep GLOBAL voxel
 * coordinates and brick ids; vr_sort_bricks lists resident bricks only; vr_render_mip / vr_render_ea
 * (one accumulator carried through all bricks) return VR_ERR_STATE.  end_brick < 0: all bricks. */
int vr_set_brick_window(vr_ctx* ctx, int first_brick, int end_brick);
int vr_window_layout(int nx, int ny, int nz, int bx, int by, int bz, int first_brick, int end_brick,
                     size_t* cube_bytes, size_t* meta_bytes);
/* Front-to-back order (O-9) of n_groups groups of bricks under the current view, group g = bricks
 * [h_group_first[g], h_group_first[g+1]) (n_groups + 1 ascending entries, whole z-layers of the
 * brick grid, covering all bricks): along any ray the z index of the bricks moves monotonically
 * away from the eye's, so slabs are met in the order of their smallest brick key, and slabs with
 * equal key never share a ray.  Folding the groups' composited partial frames in this order with
 * vr_composite_bricks equals the fold over all bricks up to float32 reassociation (MIP: exactly). */
int vr_sort_groups(vr_ctx* ctx, const int* h_group_first, int n_groups, int* h_group_order);

/* One kernel for the exchange, the fold and the gather of a sharded frame ("composite fused into the
 * exchange"; PAPER.md line 13 / line 19: images of sub-volumes rendered on distributed GPUs are composited).  Rank r
 * of n holds a full-frame partial image of its slab (vr_render_bricks + vr_composite_bricks with bg = 0, or -inf for
 * MIP) in h_d_frames[r]: DEVICE pointers to this device's memory or to a peer's, mapped into this process (CUDA IPC:
 * vr_ipc_export on the owner, vr_ipc_open here; or any peer-accessible allocation), float4 (EA) / float (MIP) pixels,
 * rows pitch_px apart.  The call folds rows [y0, y0 + rows) of the n images in the order h_order (front first, from
 * vr_sort_groups), reading each pixel straight from the owners' memory over NVLink, applies the background and stores
 * the finished rows into the same rows of every frame of h_d_out[0 .. n_out) (each rank's final frame: the gather).
 * No staging copy and no scratch.  The caller orders it after all ranks' partial frames are complete (a barrier). */
int vr_fold_peers(vr_ctx* ctx, int mode, const void* const* h_d_frames, const int* h_order, int n, int width, int height,
                  size_t pitch_px, int y0, int rows, void* const* h_d_out, int n_out, size_t out_pitch_px, const float bg[4],
                  void* stream);
/* CUDA IPC plumbing for the above: handle (64 bytes) + byte offset of d_ptr inside its allocation, to be sent to the
 * peer processes; vr_ipc_open maps it there (the mapping lives until vr_destroy). */
int vr_ipc_export(vr_ctx* ctx, const void* d_ptr, unsigned char handle[64], size_t* offset);
int vr_ipc_open(vr_ctx* ctx, const unsigned char handle[64], size_t offset, void** d_ptr);

/* ---- catalogue overlay (section 2: a source finder's
 *      output, "a set of detected astronomical sources represented by their bounding cubes",
 *      "superimposed as wireframe boxes on the volume rendering output"; "the user interaction
 *      with the displayed volume rendering output is automatically applied to the displayed source
 *      cubes"; a source can be selected; groups can be shown / hidden; catalogues can be told apart
 *      by colour).  Reading O-14 in DESIGN.md states the rasterisation rule. ------------------- */
typedef struct {
    const int* d_boxes;             /* device: n x 6 ints xlo xhi ylo yhi zlo zhi, voxel coordinates, inclusive */
    const float* d_colours;         /* device: n x 4 floats (r,g,b,a), 16-byte aligned; may be NULL if no frame is painted */
    const unsigned char* d_visible; /* device: n bytes, 0 = hidden; NULL = all shown */
    int n;
} vr_catalogue;
/* Draw the wireframes of the shown boxes under the current view into the viewport of d_pick
 * (ints, same pitch and placement as the frame: 0 = no edge, else 1 + the highest id of the boxes
 * covering the pixel; the viewport is cleared first) and, if d_frame_rgba != NULL, paint the
 * covered pixels of the frame with their box's colour (opaque, depth-unaware). */
int vr_overlay_catalogue(vr_ctx* ctx, const vr_catalogue* cat, float* d_frame_rgba, int* d_pick, void* stream);
/* The box to select for a click at view pixel (x, y): among the covered pixels of the square
 * window of half-width radius (<= 64) the one at the smallest Euclidean distance, ties to the
 * larger id; *box = -1 if none.  Synchronises `stream`. */
int vr_overlay_pick(vr_ctx* ctx, const int* d_pick, int x, int y, int radius, int* box, void* stream);

/* ---- output pyramid (section 3: "The rendering output is
 *      stored in TIFF format, which is converted to the pyramidal tiled TIFF format").  The TIFF
 *      container is the client's; this is its pixel content in a device buffer (O-15):
 *      level 0 = the frame quantised to RGBA8, q = floor(clamp(c,0,1) * 255 + 1/2); level l+1 = 2 x 2
 *      box reduction (mean of the up to 4 pixels, rounded half up), ceil(w/2) x ceil(h/2); levels
 *      until one tile holds the image; each level as tile x tile tiles (tile a power of two in
 *      [16, 4096]), row-major over the tiles, each tile contiguous, edge tiles zero padded. ------ */
#define VR_PYRAMID_MAX_LEVELS 32
typedef struct {
    int width, height;   /* pixels of the level */
    int tiles_x, tiles_y;
    size_t offset;       /* bytes from the start of the buffer to the level's first tile */
} vr_pyramid_level;
/* Sizes: levels[] needs room for VR_PYRAMID_MAX_LEVELS entries; *bytes = the whole buffer. */
int vr_pyramid_layout(int width, int height, int tile, int* n_levels, vr_pyramid_level* levels, size_t* bytes);
/* d_frame_rgba: device, float4 pixels, rows pitch_px apart (e.g. the 9600 x 5400 tiled-display
 * frame); d_out: device, *bytes of vr_pyramid_layout, caller-owned. */
int vr_build_pyramid(vr_ctx* ctx, const float* d_frame_rgba, int width, int height, size_t pitch_px, int tile,
                     void* d_out, void* stream);

/* ---- measurement of the bytes a frame needs ("B_touch = 32 B x distinct sectors inside
 *      the 2 x 2 x 2 footprints of taken samples ... measure it once per config with a debug kernel that
 *      sets one bit per sector").  Not on the frame path: bench.py and the tests call it. ------------- */
/* Bytes of the caller-owned device bitmap: one bit per 32-byte sector of the resident brick-major cube. */
int vr_touch_layout(vr_ctx* ctx, size_t* bitmap_bytes);
/* Walk the same (pixel, brick) samples as vr_render_bricks(mode, h_partials, n, ert_tau) one by one, apply
 * the skipping tests of the current plan (O-10; vr_get_plan) and early ray termination (O-7), and set the
 * bit of every sector under the 8 corners of every sample that is interpolated.  accumulate == 0 clears the
 * bitmap and the taken-sample count first (so several launches, e.g. the panels of a tiled frame, can be
 * summed or measured one by one). */
int vr_measure_touch(vr_ctx* ctx, int mode, const vr_partial* h_partials, int n, float ert_tau, void* d_bitmap,
                     int accumulate, void* stream);
/* out[0] = sectors set, out[1] = 128-byte lines with at least one sector set (the unit HBM is read in,
 * DESIGN.md section 4), out[2] = samples interpolated by the vr_measure_touch calls since the last clear.
 * Synchronises `stream`. */
int vr_touch_count(vr_ctx* ctx, const void* d_bitmap, uint64_t out[3], void* stream);

/* ---- counters (SURVEY.md section 5 "metrics") ---------------------------------------------- */
typedef struct {
    int64_t rays;             /* rays that had at least one lattice sample inside the cube */
    int64_t nominal_samples;  /* lattice samples inside the cube (O-3) */
    int64_t taken_samples;    /* samples actually interpolated (after skipping and ERT) */
    int64_t bricks_visited;   /* (ray, brick) or (ray, cell) runs marched */
    int64_t bricks_skipped;   /* runs skipped by min/max (O-10) */
    int64_t rays_terminated;  /* rays stopped by ERT */
    int64_t kernel_launches;  /* kernels launched by this context since the last reset */
} vr_counters;
/* Synchronises `stream`, then copies the device counters. */
int vr_get_counters(vr_ctx* ctx, vr_counters* out, void* stream);
int vr_reset_counters(vr_ctx* ctx, void* stream);
/* Options.  None of them but VR_OPT_VOXEL_TYPE changes a frame (tests assert it); they exist for A/B measurements.
 *  VR_OPT_SKIP (default 1): min/max empty-space skipping (O-10) on/off, all levels.
 *  VR_OPT_VARIANT (default -1): the marcher.  0 = one ray per thread, the 32 lanes of a warp take
 *    8 x 4 pixels; for partial images one CTA per pixel tile walks all bricks over the tile (ray
 *    set up once); 1 = the same with one CTA per (brick, tile); 3 = lockstep: a warp walks its 32
 *    rays together through chunks of 32 lattice indices; 4 = for dense rays,
 *    emission-absorption with occupancy bits: per chunk every lane cuts its ray into macro-cell runs, the
 *    warp then tests the samples of active runs in step, compacts, gathers and folds (any other
 *    mode / skipping level under 4 runs as 0); -1 = chosen per view from the spacing of neighbouring
 *    rays (>= 2 voxels: 3, else 4 where it applies, else 0).
 *  VR_OPT_CELL_SKIP (default -1): the 8^3 macro-cell level of the skipping under the configured
 *    bricks, 1 on / 0 off (needs VR_OPT_SKIP); -1 = on for emission-absorption if fewer than 3/4
 *    of the cells are active against the current table, on for MIP in variant 3.
 *  VR_OPT_LAYOUT (default 1): voxel order inside a brick, 0 = rows (x fastest), 1 = 4 x 4 x 2
 *    micro-blocks of one 128-byte line each; read by the next upload / generate / attach call.
 *  VR_OPT_L2_FETCH: cudaLimitMaxL2FetchGranularity of the device (32, 64 or 128 bytes; measured
 *    to have no effect on B200, where HBM is read in whole 128-byte lines).
 *  VR_OPT_DENSE (default -1): how the lockstep marcher folds emission-absorption samples, 1 =
 *    through shared memory, all rays of a warp in parallel; 0 = one by one in the lane that owns
 *    the ray; -1 = 0 if the table starts with transparent entries, else 1.
 *  VR_OPT_OCCUPANCY (default -1): the finest level of the skipping, one bit per trilinear cell,
 *    classified on the device when the set of transparent table entries changes (one pass over the
 *    cube); used by the lockstep marcher for emission-absorption with VR_OPT_DENSE 0 on layout 1.
 *    1 / -1 = on where it applies, 0 = off.
 *  VR_OPT_RING (default -1): where the lockstep marcher keeps the gathers in flight, 0 = a ring of
 *    cp.async slots in shared memory, 1 = registers; -1 = registers on layout 1 (measured faster at every
 *    view), the cp.async ring on layout 0.
 *  VR_OPT_VOXEL_TYPE (default 0): how voxels are stored in HBM (SURVEY.md 8(f)-4 "reduced-precision bricks"; PAPER.md
 *    line 19: cubes "larger than a single machine memory limit"): 0 = float32; 1 = float16, IEEE half precision,
 *    each voxel rounded to nearest even when the cube is uploaded / generated and converted back (exactly) when it is
 *    read, so the renderer computes on the cube Q(v) = float32(float16(v)) with the same float32 arithmetic (DESIGN.md
 *    O-16): half the bytes per voxel, a 256 GiB-class cube fits one B200.  Needs VR_OPT_LAYOUT 1; read by the next
 *    upload / generate / attach call; |v| beyond the float16 range (65504) is refused like a non-finite voxel.
 *    THIS option changes frames (by the quantisation of the cube, nothing else).
 *  VR_OPT_MIP_TILES (default -1): per-brick partial images by maximum intensity (vr_render_bricks / vr_render_sortlast, MIP)
 *    in OBJECT order: the bricks are cut into tiles of 32 x 32 x 16 cells that stream through shared memory (bulk
 *    asynchronous copies), every tile samples the rays that cross it and merges with an atomic maximum (MIP is order
 *    independent, the partial images are the same to the bit).  1 = on, 0 / -1 = off (the image-order marchers measured
 *    faster on every workload of bench.py: DESIGN.md section 5); float32 voxels on layout 1.  The library keeps one ray record (48 bytes)
 *    per view pixel for it, allocated at first use. */
enum { VR_OPT_SKIP = 1, VR_OPT_VARIANT = 2, VR_OPT_CELL_SKIP = 3, VR_OPT_L2_FETCH = 4, VR_OPT_LAYOUT = 5, VR_OPT_DENSE = 6,
       VR_OPT_OCCUPANCY = 7, VR_OPT_RING = 8, VR_OPT_VOXEL_TYPE = 9, VR_OPT_MIP_TILES = 10 };
int vr_set_option(vr_ctx* ctx, int option, int value);
/* What a render call of `mode` would launch under the current cube, view and transfer function:
 * out[0] = marcher variant (0 / 3 / 4; 5 = the object-order MIP of VR_OPT_MIP_TILES), out[1] = skipping level of the sort-last path, vr_render_bricks / vr_render_sortlast
 * (0 none, 1 bricks, 2 + macro-cells, 3 + occupancy bits; the whole-frame vr_render_mip, which carries one maximum
 * through all bricks, also uses the macro-cells where the sort-last MIP stops at the brick level),
 * out[2] = VR_OPT_DENSE as resolved (0 / 1).  May classify the cube against
 * the table (as the render call would) and then synchronises `stream`. */
int vr_get_plan(vr_ctx* ctx, int mode, int out[3], void* stream);

#ifdef __cplusplus
}
#endif
#endif
