// Internal declarations shared by the libvr translation units (not part of the C ABI).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <string>
#include <vector>

#include "../../include/vr.h"

namespace vr {

constexpr int kCell = 8;            // edge of the min/max macro-cells under the configured bricks
constexpr int kTileW = 16, kTileH = 8, kThreads = 128;   // pixel tile of one CTA: 4 warps of 8x4

// Brick-major cube in HBM.  Brick b = bx + G0 (by + G1 bz) occupies
// `stride` floats; it stores voxels (lx,ly,lz), 0 <= l <= B (the +1 is the one-sided halo).
// Halo voxels beyond the cube and padding slots are zero.  Two layouts inside a brick:
//  layout 0 (rows):   offset = lx + P0 (ly + P1 lz), P0 = roundup4(B0 + 1);
//  layout 1 (blocks): 4 x 4 x 2 micro-blocks of 32 voxels = one 128-byte line each,
//                     offset = 32 ((lx>>2) + T0 ((ly>>2) + T1 (lz>>1)))
//                              + 16 ((ly>>1)&1) + 8 (lz&1) + 4 (ly&1) + (lx&3),
//                     i.e. a 32-byte sector is 4 x 2 x 1 voxels and each 64-byte half line (the
//                     unit HBM is read in) is 4 x 2 x 2, so that a ray's 2 x 2 x 2 footprints
//                     meet about the same, small number of lines and half lines whatever its
//                     direction.
struct CubeDesc {
    int N[3];        // voxels
    int B[3];        // configured brick size
    int G[3];        // brick grid
    int P[3];        // stored brick extents: B + 1 (layout 0: P0 rounded up to a multiple of 4)
    int layout;      // 0: rows, 1: 4x4x2 micro-blocks
    int vtype;       // stored voxel type: 0 float32, 1 float16 (IEEE half, layout 1 only); `stride` counts voxels
    int T[3];        // layout 1: micro-blocks per axis = ceil(P0/4), ceil(P1/4), ceil(P2/2)
    int sh[3];       // log2(B) if B is a power of two, else -1
    int C[3];        // macro-cells per brick axis = ceil(B / kCell)
    int nbricks;
    int win_lo, win_hi;          // resident bricks [win_lo, win_hi) (all by default); the pointers below are
                                 // shifted so that GLOBAL brick ids index them (vr_set_brick_window)
    int cells_per_brick;
    long long stride;            // voxels per brick (multiple of 32)
    const float* cube;
    float2* brick_mm;            // (min,max) per brick, halo-inclusive
    float2* cell_mm;             // (min,max) per macro-cell, halo-inclusive, brick-major
    unsigned* cell_bits;         // EA activity of macro-cells vs the transfer function, 1 bit each
    int* brick_active;           // EA activity of bricks vs the transfer function
    int cell_words_per_brick;
    // Occupancy bits (layout 1 only): one bit per trilinear cell (lower corner (lx,ly,lz), l < B), set iff one of
    // its 8 corners maps above the transparent prefix of the table (O-10 at the finest level).  One 32-bit word per
    // 4 x 4 x 2 micro-block, in the order of the block's 128-byte line in the brick (word = line index), bit = the
    // slot of the lower corner inside the line, (lx&3) + 4 (ly&1) + 8 (lz&1) + 16 ((ly>>1)&1).
    unsigned* occ;
    unsigned* hot;               // scratch of the same shape: one bit per VOXEL ("maps above the transparent prefix")
    int occ_words_per_brick;     // T0 T1 T2
};

struct ViewDesc {
    double Minv[16];
    int W, H;
    float step;
    int vx0, vy0;
    long long pitch;
};

struct TFDesc {
    const float4* baked;   // device: opacity-corrected table (O-6)
    const float4* raw;     // device: raw table
    float vmin, scale;     // scale = (float)(255 / (vmax - vmin))
    float x_clear;         // table coordinates below it lie between entries of zero baked opacity
};

struct PartialDev {        // device descriptor of one partial image
    int brick, x0, y0, w, h, tile0;   // tile0: first CTA tile of this partial in the launch
    long long pitch;
    void* data;
    int b[3];                         // the brick's grid coordinates (brick = b0 + G0 (b1 + G1 b2)), so that no kernel divides
    int otile0;                       // first object tile of this brick in a mip_tiles_kernel launch (vr_mip_tiles.cu)
};
inline void set_brick(PartialDev& d, const CubeDesc& c, int brick) {
    d.brick = brick; d.otile0 = 0;
    if (brick >= 0 && c.G[0] > 0 && c.G[1] > 0) { d.b[0] = brick % c.G[0]; d.b[1] = (brick / c.G[0]) % c.G[1]; d.b[2] = brick / (c.G[0] * c.G[1]); }
    else d.b[0] = d.b[1] = d.b[2] = 0;
}

enum Counter { kRays = 0, kNominal, kTaken, kVisited, kSkipped, kTerminated, kNumCounters };

// offset (floats) of stored voxel (lx, ly, lz) inside its brick
__host__ __device__ inline long long voxel_slot(const CubeDesc& c, int lx, int ly, int lz) {
    if (c.layout == 0) return lx + (long long)c.P[0] * (ly + (long long)c.P[1] * lz);
    return 32LL * ((lx >> 2) + (long long)c.T[0] * ((ly >> 2) + (long long)c.T[1] * (lz >> 1))) +
           16 * ((ly >> 1) & 1) + 8 * (lz & 1) + 4 * (ly & 1) + (lx & 3);
}

size_t align_up(size_t v, size_t a);
void fill_cube_desc(CubeDesc& c, int nx, int ny, int nz, int bx, int by, int bz, int layout, int vtype = 0);
size_t cube_bytes(const CubeDesc& c);
struct MetaLayout { size_t brick_mm, cell_mm, cell_bits, brick_active, occ, hot, total; };
MetaLayout meta_layout(const CubeDesc& c);

// kernels' host launchers (vr_cube.cu / vr_march.cu / vr_composite.cu)
cudaError_t launch_rebrick(const CubeDesc& c, float* d_cube, const float* d_src, int z0, int z1, unsigned long long* d_bad,
                           cudaStream_t s);
cudaError_t launch_unbrick(const CubeDesc& c, int brick, float* d_dst, cudaStream_t s);
cudaError_t launch_minmax(const CubeDesc& c, cudaStream_t s);
struct GenDev {
    const double* sources; const int* tile_offsets; const int* tile_ids; int tiles[3];
    const int* zero_boxes; int n_zero; double continuum; uint64_t seed;
};
cudaError_t launch_generate(const CubeDesc& c, float* d_cube, const GenDev& g, cudaStream_t s);

struct RenderArgs {
    int mode; float tau; float bg[4]; float miss;
    int skip;              // 0: none; 1: configured bricks; 2: + 8^3 macro-cells; 3: + occupancy bits (O-10)
    int variant;           // 0: one ray per thread; 3: lockstep (the lanes of a warp take one ray's samples)
    int ring;              // lockstep marcher: 0 gathers through the cp.async ring in shared memory, 1 through registers
    int dense;             // lockstep EA: fold through shared memory, all rays in parallel (see vr_march.cu)
    float* out; float* out_rgba; unsigned long long* counters;
};
cudaError_t launch_render_global(const CubeDesc& c, const ViewDesc& v, const TFDesc& t, const RenderArgs& a, cudaStream_t s);
cudaError_t launch_render_bricks(const CubeDesc& c, const ViewDesc& v, const TFDesc& t, const RenderArgs& a,
                                 const PartialDev* d_partials, int n, int total_tiles, cudaStream_t s);
// object-order MIP of per-brick partial images (vr_mip_tiles.cu)
int object_tiles_of_brick(const CubeDesc& c, const int b[3]);
size_t ray_buffer_bytes(int W, int H);
cudaError_t launch_mip_tiles(const CubeDesc& c, const ViewDesc& v, const double M[16], const RenderArgs& a, const PartialDev* d_partials,
                             int n, int total_pixel_tiles, int total_object_tiles, float4* d_rays, cudaStream_t s);
cudaError_t launch_touch(const CubeDesc& c, const ViewDesc& v, const TFDesc& t, const RenderArgs& a, const PartialDev* d_partials,
                         int n, int total_tiles, unsigned* d_bitmap, unsigned long long* d_taken, cudaStream_t s);
cudaError_t launch_touch_count(const unsigned* d_bitmap, long long n_words, unsigned long long* d_out, cudaStream_t s);
cudaError_t launch_composite(const ViewDesc& v, int mode, const PartialDev* d_partials, int n, float* out,
                             const float bg[4], cudaStream_t s);
// vr_composite_bricks_static (vr_composite_static.cu): the descriptors live in a static __device__ array of the library
constexpr int kStaticMaxPartials = VR_STATIC_MAX_PARTIALS;
cudaError_t static_partials_store(int first, const PartialDev* h, int count, cudaStream_t s);
cudaError_t launch_composite_static(const ViewDesc& v, int mode, int n, float* out, const float bg[4], cudaStream_t s);
constexpr int kMaxPeers = 32;
struct PeerList { const void* in[kMaxPeers]; void* out[kMaxPeers]; int n, n_out; };   // `in` already in fold order
cudaError_t launch_fold_peers(const PeerList& L, int mode, int width, long long pitch, int y0, int rows, long long out_pitch,
                              const float bg[4], cudaStream_t s);
cudaError_t launch_classify_cells(const CubeDesc& c, const int nz_prefix[257], float vmin, float scale,
                                  unsigned long long* d_active_count, cudaStream_t s);
cudaError_t launch_classify_occ(const CubeDesc& c, float vmin, float scale, float thr, cudaStream_t s);
cudaError_t launch_cell_minmax_lines(const CubeDesc& c, cudaStream_t s);
cudaError_t launch_overlay(const ViewDesc& v, const double M[16], const int* d_boxes, const float* d_colours,
                           const unsigned char* d_visible, int n, float* d_frame, int* d_pick, cudaStream_t s);
cudaError_t launch_overlay_pick(const ViewDesc& v, const int* d_pick, int x, int y, int radius, int* d_out, cudaStream_t s);
int pyramid_levels(int width, int height, int tile, vr_pyramid_level* lv, size_t* bytes);
cudaError_t launch_pyramid(const float* d_frame, int width, int height, long long pitch, int tile, void* d_out, int* launches,
                           cudaStream_t s);
cudaError_t launch_upload_table(float4* d_dst, const float* h_src_1024, cudaStream_t s);

}  // namespace vr
