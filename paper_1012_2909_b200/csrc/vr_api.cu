// Host side of libvr: the C ABI of include/vr.h.  Per-view / per-transfer-function setup
// (matrix inverse in fp64, opacity-corrected table, brick classification
// against the table, visibility keys + sort) and the launch plumbing.  No torch types.
#ifndef VR_PIN_SLOTS
#define VR_PIN_SLOTS 32   // descriptor slots of vr_render_sortlast (calls the host may have in flight)
#endif
#include <algorithm>
#include <climits>
#include <cmath>
#include <cstdio>
#include <cstring>

#include <cuda.h>
#include <nvtx3/nvToolsExt.h>

#include "vr_internal.cuh"

using namespace vr;

// One corner of a brick under the current view: NDC coordinates, or `behind` (w <= 0: no projection).
struct Corner { double xn, yn, zn; bool behind; };

struct vr_ctx {
    int device = 0;
    std::string err;
    // cube
    bool has_cube = false;
    CubeDesc cube{};
    std::vector<float2> h_brick_mm;
    // view
    bool has_view = false;
    double M[16], Minv[16];
    ViewDesc view{};
    // transfer function
    bool has_tf = false;
    float tf_raw[1024], tf_baked[1024];
    float vmin = 0, vmax = 1, scale = 1;
    float baked_step = -1;
    bool tables_dirty = true, activity_dirty = true;
    std::vector<int> h_brick_active;
    // small device scratch owned by the library
    float4* d_tf_baked = nullptr;
    float4* d_tf_raw = nullptr;
    unsigned long long* d_counters = nullptr;
    PartialDev* d_partials = nullptr;
    size_t partials_cap = 0;
    int64_t launches = 0;
    int opt_skip = 1, opt_cell_skip = -1, opt_variant = -1, opt_layout = 1, opt_dense = -1, opt_occ = -1, opt_ring = -1;   // -1: chosen per view / TF
    int opt_mip_tiles = -1;
    // object-order MIP (vr_mip_tiles.cu): one ray record per view pixel, one buffer per descriptor slot of
    // vr_render_sortlast (calls in flight on different streams) plus one for vr_render_bricks; grown on demand
    static constexpr int kPinSlots = VR_PIN_SLOTS;
    float4* d_rays[kPinSlots + 1] = {};
    size_t rays_bytes[kPinSlots + 1] = {};
    int opt_vtype = 0;                   // VR_OPT_VOXEL_TYPE: 0 float32, 1 float16
    float x_clear = -INFINITY;
    double active_cell_fraction = 1.0;   // macro-cells active against the current table (EA)
    unsigned long long* d_scratch = nullptr;
    // what the activity bits on the device (bricks, macro-cells, occupancy) were classified against:
    // the zero pattern of the baked opacities and the value -> table mapping
    bool key_valid = false, occ_valid = false;
    int key_nz[257];
    float key_vmin = 0, key_scale = 0;
    int win_lo = 0, win_hi = -1;         // vr_set_brick_window (hi < 0: all bricks)
    std::vector<void*> ipc_bases;        // peer allocations opened by vr_ipc_open
    // vr_render_sortlast: descriptors staged through a small ring of pinned slots (no allocation, no pageable copy per frame)
    // (32 slots: the host may run a whole tiled frame of 25 panels ahead of the GPU; with 4 it stalled at every frame start
    // until the GPU had finished the last panels of the frame before: C4 end to end 19.9 ms against 17.5 on the device)
    PartialDev* h_pin = nullptr;
    PartialDev* d_pin = nullptr;         // the same slots on the device: calls on different streams do not share descriptors
    size_t pin_cap = 0;                  // descriptors per slot
    cudaEvent_t pin_done[kPinSlots] = {};
    int pin_next = 0;
    std::vector<std::pair<int, int>> keyed;   // scratch: (visibility key, brick)
    std::vector<int> key_count;               // scratch of the counting sort in vr_render_sortlast
    std::vector<Corner> corner_grid;          // scratch: the brick grid's corners under the current view
    std::vector<int> keys;
};

namespace {

// One NVTX range per C-ABI call that does work (SURVEY.md section 5 "tracing"): an nsys trace of an orbit then reads
// as set_view / sort / render / composite per frame.  Header-only NVTX: a no-op unless a profiler is attached.
struct Range {
    explicit Range(const char* name) { nvtxRangePushA(name); }
    ~Range() { nvtxRangePop(); }
};
#define VR_RANGE() Range nvtx_range__(__func__)

constexpr double kSparseRaySpacing = 2.0;     // voxels between neighbouring rays: variant 3 at or above
constexpr double kCellSkipMaxActive = 0.75;   // macro-cell skipping only if fewer cells than this are active

int fail(vr_ctx* ctx, int code, const std::string& msg) {
    if (ctx) ctx->err = msg;
    return code;
}

int cuda_fail(vr_ctx* ctx, cudaError_t e, const char* where) {
    return fail(ctx, VR_ERR_CUDA, std::string(where) + ": " + cudaGetErrorString(e));
}

#define VR_CUDA(ctx, call)                                             \
    do {                                                               \
        cudaError_t e__ = (call);                                      \
        if (e__ != cudaSuccess) return cuda_fail(ctx, e__, #call);     \
    } while (0)

// 4x4 inverse by cofactors (adjugate / determinant), fp64.  The expansion below is the textbook closed
// form in the term order of the widely circulated Mesa GLU listing (gluInvertMatrix); the oracle
// inverts with an independent Gauss-Jordan elimination (oracle/ovr.cpp).
bool invert4(const double m[16], double inv[16]) {
    double a[16];
    a[0] = m[5] * m[10] * m[15] - m[5] * m[11] * m[14] - m[9] * m[6] * m[15] + m[9] * m[7] * m[14] + m[13] * m[6] * m[11] - m[13] * m[7] * m[10];
    a[4] = -m[4] * m[10] * m[15] + m[4] * m[11] * m[14] + m[8] * m[6] * m[15] - m[8] * m[7] * m[14] - m[12] * m[6] * m[11] + m[12] * m[7] * m[10];
    a[8] = m[4] * m[9] * m[15] - m[4] * m[11] * m[13] - m[8] * m[5] * m[15] + m[8] * m[7] * m[13] + m[12] * m[5] * m[11] - m[12] * m[7] * m[9];
    a[12] = -m[4] * m[9] * m[14] + m[4] * m[10] * m[13] + m[8] * m[5] * m[14] - m[8] * m[6] * m[13] - m[12] * m[5] * m[10] + m[12] * m[6] * m[9];
    a[1] = -m[1] * m[10] * m[15] + m[1] * m[11] * m[14] + m[9] * m[2] * m[15] - m[9] * m[3] * m[14] - m[13] * m[2] * m[11] + m[13] * m[3] * m[10];
    a[5] = m[0] * m[10] * m[15] - m[0] * m[11] * m[14] - m[8] * m[2] * m[15] + m[8] * m[3] * m[14] + m[12] * m[2] * m[11] - m[12] * m[3] * m[10];
    a[9] = -m[0] * m[9] * m[15] + m[0] * m[11] * m[13] + m[8] * m[1] * m[15] - m[8] * m[3] * m[13] - m[12] * m[1] * m[11] + m[12] * m[3] * m[9];
    a[13] = m[0] * m[9] * m[14] - m[0] * m[10] * m[13] - m[8] * m[1] * m[14] + m[8] * m[2] * m[13] + m[12] * m[1] * m[10] - m[12] * m[2] * m[9];
    a[2] = m[1] * m[6] * m[15] - m[1] * m[7] * m[14] - m[5] * m[2] * m[15] + m[5] * m[3] * m[14] + m[13] * m[2] * m[7] - m[13] * m[3] * m[6];
    a[6] = -m[0] * m[6] * m[15] + m[0] * m[7] * m[14] + m[4] * m[2] * m[15] - m[4] * m[3] * m[14] - m[12] * m[2] * m[7] + m[12] * m[3] * m[6];
    a[10] = m[0] * m[5] * m[15] - m[0] * m[7] * m[13] - m[4] * m[1] * m[15] + m[4] * m[3] * m[13] + m[12] * m[1] * m[7] - m[12] * m[3] * m[5];
    a[14] = -m[0] * m[5] * m[14] + m[0] * m[6] * m[13] + m[4] * m[1] * m[14] - m[4] * m[2] * m[13] - m[12] * m[1] * m[6] + m[12] * m[2] * m[5];
    a[3] = -m[1] * m[6] * m[11] + m[1] * m[7] * m[10] + m[5] * m[2] * m[11] - m[5] * m[3] * m[10] - m[9] * m[2] * m[7] + m[9] * m[3] * m[6];
    a[7] = m[0] * m[6] * m[11] - m[0] * m[7] * m[10] - m[4] * m[2] * m[11] + m[4] * m[3] * m[10] + m[8] * m[2] * m[7] - m[8] * m[3] * m[6];
    a[11] = -m[0] * m[5] * m[11] + m[0] * m[7] * m[9] + m[4] * m[1] * m[11] - m[4] * m[3] * m[9] - m[8] * m[1] * m[7] + m[8] * m[3] * m[5];
    a[15] = m[0] * m[5] * m[10] - m[0] * m[6] * m[9] - m[4] * m[1] * m[10] + m[4] * m[2] * m[9] + m[8] * m[1] * m[6] - m[8] * m[2] * m[5];
    double det = m[0] * a[0] + m[1] * a[4] + m[2] * a[8] + m[3] * a[12];
    if (det == 0.0 || !std::isfinite(det)) return false;
    for (int i = 0; i < 16; ++i) {
        inv[i] = a[i] / det;
        if (!std::isfinite(inv[i])) return false;
    }
    return true;
}

bool valid_dims(int nx, int ny, int nz, int bx, int by, int bz) {
    if (!(nx > 0 && ny > 0 && nz > 0 && bx > 0 && by > 0 && bz > 0 &&
          (long long)nx < (1 << 22) && (long long)ny < (1 << 22) && (long long)nz < (1 << 22))) return false;
    // brick ids, cells per brick and occupancy words per brick are ints: bound them (2^24 bricks, 2^26 cells)
    const int N[3] = {nx, ny, nz}, B[3] = {std::min(bx, nx), std::min(by, ny), std::min(bz, nz)};
    long long bricks = 1, cells = 1;
    for (int a = 0; a < 3; ++a) { bricks *= (N[a] + B[a] - 1) / B[a]; cells *= (B[a] + kCell - 1) / kCell + 1; }
    return bricks <= (1LL << 24) && cells <= (1LL << 26);
}

// Point the descriptor at the caller's buffers.  They hold the bricks of the window only; every
// pointer is shifted back by the window's first brick so that global brick ids index it.
void bind_meta(CubeDesc& c, const void* d_cube, void* d_meta) {
    MetaLayout ml = meta_layout(c);
    char* m = (char*)d_meta;
    const long long lo = c.win_lo;
    c.cube = c.vtype == 1 ? (const float*)((const unsigned short*)d_cube - lo * c.stride) : (const float*)d_cube - lo * c.stride;
    c.brick_mm = (float2*)(m + ml.brick_mm) - lo;
    c.cell_mm = (float2*)(m + ml.cell_mm) - lo * c.cells_per_brick;
    c.cell_bits = (unsigned*)(m + ml.cell_bits) - lo * c.cell_words_per_brick;
    c.brick_active = (int*)(m + ml.brick_active) - lo;
    c.occ = (unsigned*)(m + ml.occ) - lo * c.occ_words_per_brick;
    c.hot = (unsigned*)(m + ml.hot) - lo * c.occ_words_per_brick;
}

void apply_window(const vr_ctx* ctx, CubeDesc& c) {
    if (ctx->win_hi >= 0) { c.win_lo = std::min(ctx->win_lo, c.nbricks); c.win_hi = std::min(ctx->win_hi, c.nbricks); }
}

// (min,max) of the resident bricks to the host; bricks outside the window read as empty
int fetch_brick_mm(vr_ctx* ctx, cudaStream_t s) {
    const CubeDesc& c = ctx->cube;
    ctx->h_brick_mm.assign(c.nbricks, make_float2(INFINITY, -INFINITY));
    if (c.win_hi > c.win_lo)
        VR_CUDA(ctx, cudaMemcpyAsync(ctx->h_brick_mm.data() + c.win_lo, c.brick_mm + c.win_lo, sizeof(float2) * (c.win_hi - c.win_lo),
                                     cudaMemcpyDeviceToHost, s));
    VR_CUDA(ctx, cudaStreamSynchronize(s));
    return VR_OK;
}

int finish_cube(vr_ctx* ctx, cudaStream_t s) {
    CubeDesc& c = ctx->cube;
    if (c.win_hi > c.win_lo) {                              // an empty window (more ranks than brick layers) launches nothing
        VR_CUDA(ctx, launch_minmax(c, s));
        ctx->launches += 2;
    }
    int rc = fetch_brick_mm(ctx, s);
    if (rc) return rc;
    ctx->has_cube = true;
    ctx->activity_dirty = true; ctx->key_valid = false; ctx->occ_valid = false;
    return VR_OK;
}

// O-6: a'_i = 1 - (1 - a_i)^Delta in fp64, rounded to float32; colours unchanged.
void bake_tf(vr_ctx* ctx) {
    const double step = (double)ctx->view.step;
    for (int i = 0; i < 256; ++i) {
        for (int ch = 0; ch < 3; ++ch) ctx->tf_baked[4 * i + ch] = ctx->tf_raw[4 * i + ch];
        ctx->tf_baked[4 * i + 3] = (float)(1.0 - std::pow(1.0 - (double)ctx->tf_raw[4 * i + 3], step));
    }
    ctx->baked_step = ctx->view.step;
}

// O-10: a brick is inactive iff a'_j = 0 for every table index the values of [min, max] can
// touch, j in [floor(x(min)), ceil(x(max))], x evaluated exactly as the kernel evaluates it.
bool range_active(const vr_ctx* ctx, float mn, float mx) {
    if (!(mn <= mx)) return false;                           // empty brick (no voxel of the cube)
    auto xof = [&](float v) {
        float x = (v - ctx->vmin) * ctx->scale;
        return std::fmin(std::fmax(x, 0.f), 255.f);
    };
    int lo = (int)std::floor(xof(mn)), hi = (int)std::ceil(xof(mx));
    lo = std::max(0, std::min(lo, 255)); hi = std::max(0, std::min(hi, 255));
    for (int j = lo; j <= hi; ++j) if (ctx->tf_baked[4 * j + 3] != 0.f) return true;
    return false;
}

int ensure_tables(vr_ctx* ctx, cudaStream_t s) {
    if (!ctx->has_tf) return VR_OK;
    if (ctx->tables_dirty || ctx->baked_step != ctx->view.step) {
        bake_tf(ctx);
        VR_CUDA(ctx, launch_upload_table(ctx->d_tf_baked, ctx->tf_baked, s));
        VR_CUDA(ctx, launch_upload_table(ctx->d_tf_raw, ctx->tf_raw, s));
        ctx->launches += 4;
        ctx->tables_dirty = false;
        ctx->activity_dirty = true;
    }
    if (ctx->activity_dirty && ctx->has_cube) {
        int nz[257];
        nz[0] = 0;
        for (int j = 0; j < 256; ++j) nz[j + 1] = nz[j] + (ctx->tf_baked[4 * j + 3] != 0.f ? 1 : 0);
        const bool same = ctx->key_valid && ctx->key_vmin == ctx->vmin && ctx->key_scale == ctx->scale &&
                          std::memcmp(nz, ctx->key_nz, sizeof(nz)) == 0;
        if (!same) {                                        // else: colours / opacities changed, not what is transparent
            const int nb = ctx->cube.nbricks;
            ctx->h_brick_active.resize(nb);
            for (int b = 0; b < nb; ++b)
                ctx->h_brick_active[b] = range_active(ctx, ctx->h_brick_mm[b].x, ctx->h_brick_mm[b].y) ? 1 : 0;
            // pageable source: cudaMemcpyAsync stages it before returning, so the vector may change later
            const int w0 = ctx->cube.win_lo, wn = ctx->cube.win_hi - ctx->cube.win_lo;
            if (wn > 0) VR_CUDA(ctx, cudaMemcpyAsync(ctx->cube.brick_active + w0, ctx->h_brick_active.data() + w0, sizeof(int) * wn, cudaMemcpyHostToDevice, s));
            // the same test per 8^3 macro-cell, on the device (one bit per cell)
            VR_CUDA(ctx, cudaMemsetAsync(ctx->d_scratch, 0, sizeof(unsigned long long), s));
            if (wn > 0) {
                VR_CUDA(ctx, launch_classify_cells(ctx->cube, nz, ctx->vmin, ctx->scale, ctx->d_scratch, s));
                ctx->launches += 1;
            }
            unsigned long long n_active = 0;
            VR_CUDA(ctx, cudaMemcpyAsync(&n_active, ctx->d_scratch, sizeof(n_active), cudaMemcpyDeviceToHost, s));
            VR_CUDA(ctx, cudaStreamSynchronize(s));
            ctx->active_cell_fraction = (double)n_active / std::max(1.0, (double)(ctx->cube.win_hi - ctx->cube.win_lo) * ctx->cube.cells_per_brick);
            std::memcpy(ctx->key_nz, nz, sizeof(nz));
            ctx->key_vmin = ctx->vmin; ctx->key_scale = ctx->scale;
            ctx->key_valid = true; ctx->occ_valid = false;
        }
        // samples with table coordinate x < x_clear interpolate two entries of zero opacity
        int i0 = -1;
        while (i0 + 1 < 256 && ctx->tf_baked[4 * (i0 + 1) + 3] == 0.f) ++i0;
        ctx->x_clear = i0 >= 1 ? (float)i0 : -INFINITY;
        ctx->activity_dirty = false;
    }
    return VR_OK;
}

// Distance in voxels between the rays of neighbouring pixels where they pass the cube centre.
double ray_spacing(const vr_ctx* ctx) {
    const CubeDesc& c = ctx->cube;
    const double* M = ctx->M; const double* Mi = ctx->Minv;
    const double ctr[3] = {0.5 * (c.N[0] - 1), 0.5 * (c.N[1] - 1), 0.5 * (c.N[2] - 1)};
    const double Z = M[8] * ctr[0] + M[9] * ctr[1] + M[10] * ctr[2] + M[11];
    const double Wc = M[12] * ctr[0] + M[13] * ctr[1] + M[14] * ctr[2] + M[15];
    const double zn = Wc > 1e-12 ? std::min(1.0, std::max(-1.0, Z / Wc)) : 0.0;
    auto unproj = [&](double xn, double yn, double out[3]) {
        double v[4];
        for (int r = 0; r < 4; ++r) v[r] = Mi[4 * r] * xn + Mi[4 * r + 1] * yn + Mi[4 * r + 2] * zn + Mi[4 * r + 3];
        for (int a = 0; a < 3; ++a) out[a] = v[a] / v[3];
    };
    double p0[3], p1[3], p2[3];
    unproj(0.0, 0.0, p0); unproj(2.0 / ctx->view.W, 0.0, p1); unproj(0.0, 2.0 / ctx->view.H, p2);
    double sx = 0, sy = 0;
    for (int a = 0; a < 3; ++a) { sx += (p1[a] - p0[a]) * (p1[a] - p0[a]); sy += (p2[a] - p0[a]) * (p2[a] - p0[a]); }
    const double s = std::sqrt(std::sqrt(sx) * std::sqrt(sy));
    return std::isfinite(s) ? s : 1.0;
}

// Marcher variant.  Rays of neighbouring pixels less than about two voxels
// apart share their cache lines inside a warp of 8 x 4 pixels: one ray per thread (variant 0).
// Sparser rays share nothing: the lanes of a warp take consecutive samples of one ray (variant 3).
int resolve_variant(const vr_ctx* ctx) {
    if (ctx->opt_variant >= 0) return ctx->opt_variant;
    return ray_spacing(ctx) >= kSparseRaySpacing ? 3 : 0;
}

int resolve_dense(const vr_ctx* ctx);

// Skipping level: 0 none, 1 configured bricks, 2 + 8^3 macro-cells, 3 + occupancy bits per trilinear
// cell.  The macro-cell level costs a lookup per run / sample, so by default emission-absorption uses
// it only if the current table leaves a fair share of the cells idle, and MIP only in the lockstep
// marcher (measured).  Level 3 serves emission-absorption with sparse tables on the micro-block layout
// (in the lockstep marcher: the test-compact-gather-fold kernel; ray per thread: a bit test per sample
// inside active macro-cells).
int skip_level(const vr_ctx* ctx, int mode, bool sortlast = false) {
    if (!ctx->opt_skip) return 0;
    if (ctx->opt_cell_skip == 0) return 1;
    if (mode == VR_MODE_EA && ctx->opt_occ != 0 && ctx->cube.layout == 1 && !resolve_dense(ctx)) return 3;
    if (ctx->opt_cell_skip > 0) return 2;
    // MIP: the macro-cell test pays where the running maximum is carried through the whole cube (vr_render_mip); a
    // per-brick partial image restarts from -inf in every brick, the test then skips 7 % of the samples of a noise cube
    // and costs a dependent load per sample (C3: 14.6 -> 13.6 ms without it): the brick-level exit serves there
    if (mode == VR_MODE_MIP) return (resolve_variant(ctx) == 3 && !sortlast) ? 2 : 1;
    return ctx->active_cell_fraction < kCellSkipMaxActive ? 2 : 1;
}

// The marcher of a render call of `mode` at skipping level `skip`: with dense rays, emission-absorption through
// a sparse table on the micro-block layout goes to variant 4 (macro-cell runs first, then the occupancy test in step
// over the warp, compaction, gather, fold), everything else of variant 0 stays a ray per thread.
int pick_variant(const vr_ctx* ctx, int mode, int skip) {
    const int v = resolve_variant(ctx);
    // small bricks: a ray spends one or two groups of chunks in a brick, the per-(tile, brick) set-up of the warp-wide
    // marcher then outweighs what it saves (C2, 64^3 bricks: 0.73 ms as variant 0, 0.80 as 4)
    const int bmin = std::min(ctx->cube.B[0], std::min(ctx->cube.B[1], ctx->cube.B[2]));
    if (v == 0 && ctx->opt_variant < 0 && mode == VR_MODE_EA && skip >= 3 && ctx->cube.layout == 1 && bmin >= 128) return 4;
    return v;
}

// Occupancy bits are classified when a render first needs them for the current table.
int ensure_occ(vr_ctx* ctx, int skip, cudaStream_t s) {
    if (skip < 3 || ctx->occ_valid) return VR_OK;
    if (ctx->cube.win_hi <= ctx->cube.win_lo) { ctx->occ_valid = true; return VR_OK; }
    // the table's transparent prefix 0 .. t: a cell whose 8 corners all map to x <= t only meets entries of zero opacity
    int t = -1;
    while (t + 1 < 256 && ctx->key_nz[t + 2] == 0) ++t;
    VR_CUDA(ctx, launch_classify_occ(ctx->cube, ctx->key_vmin, ctx->key_scale, (float)t, s));
    ctx->launches += 2;
    ctx->occ_valid = true;
    return VR_OK;
}

// Lockstep emission-absorption: fold through shared memory with all rays in parallel (dense) or
// hand the few samples above x_clear to the owning lane one by one (sparse).  By default dense
// unless the table starts with a run of transparent entries (x_clear >= 1).
int resolve_dense(const vr_ctx* ctx) {
    if (ctx->opt_dense >= 0) return ctx->opt_dense;
    return ctx->x_clear >= 1.f ? 0 : 1;
}

// Lockstep marcher: gathers through registers (1) or through the cp.async ring in shared memory (0).
// Measured over the C3 orbit with the final build (vr_march.cuh, REGS): the register ring is faster whatever the view, for
// MIP (12.9 vs 15.2 ms, mean of 12 azimuths) and, since its emission-absorption instantiations take six CTAs per SM, for
// emission-absorption with a dense table too (along x, where the cp.async ring used to win: 15.1 vs 16.0 ms; at 60 degrees
// from x 16.6 vs 19.9).  The cp.async ring serves the row layout and VR_OPT_RING 0.
int resolve_ring(const vr_ctx* ctx, int mode) {
    (void)mode;
    if (ctx->cube.vtype == 1) return 1;                      // float16 voxels: plain loads only (vr_march_h.cu)
    if (ctx->opt_ring >= 0) return ctx->opt_ring;
    return ctx->cube.layout == 1 ? 1 : 0;
}

TFDesc tf_desc(const vr_ctx* ctx) {
    TFDesc t;
    t.baked = ctx->d_tf_baked; t.raw = ctx->d_tf_raw; t.vmin = ctx->vmin; t.scale = ctx->scale;
    t.x_clear = ctx->x_clear;
    return t;
}

inline Corner project_corner(const double* M, double x, double y, double z) {
    Corner k{0.0, 0.0, 0.0, false};
    const double X = M[0] * x + M[1] * y + M[2] * z + M[3];
    const double Y = M[4] * x + M[5] * y + M[6] * z + M[7];
    const double Z = M[8] * x + M[9] * y + M[10] * z + M[11];
    const double Wc = M[12] * x + M[13] * y + M[14] * z + M[15];
    if (!(Wc > 1e-9)) { k.behind = true; return k; }
    k.xn = X / Wc; k.yn = Y / Wc; k.zn = Z / Wc;
    return k;
}

// Screen rectangle (view pixels, clipped) that holds every pixel whose ray can meet a brick with these 8 corners.
// Returns false if the brick is outside the frustum.
inline bool rect_of_corners(int W, int H, const Corner* const k[8], int rect[4]) {
    double xmin = 1e300, xmax = -1e300, ymin = 1e300, ymax = -1e300, zmin = 1e300, zmax = -1e300;
    bool behind = false;
    for (int i = 0; i < 8; ++i) {
        if (k[i]->behind) { behind = true; continue; }
        xmin = std::min(xmin, k[i]->xn); xmax = std::max(xmax, k[i]->xn);
        ymin = std::min(ymin, k[i]->yn); ymax = std::max(ymax, k[i]->yn);
        zmin = std::min(zmin, k[i]->zn); zmax = std::max(zmax, k[i]->zn);
    }
    int x0 = 0, x1 = W - 1, y0 = 0, y1 = H - 1;
    if (!behind) {
        if (zmin > 1.0 + 1e-6 || zmax < -1.0 - 1e-6) return false;      // beyond far / before near
        // pixel centre i has xn = 2 (i + 1/2) / W - 1 ; row j has yn = 1 - 2 (j + 1/2) / H
        x0 = std::max(0, (int)std::floor((xmin + 1.0) * 0.5 * W - 0.5) - 1);
        x1 = std::min(W - 1, (int)std::ceil((xmax + 1.0) * 0.5 * W - 0.5) + 1);
        y0 = std::max(0, (int)std::floor((1.0 - ymax) * 0.5 * H - 0.5) - 1);
        y1 = std::min(H - 1, (int)std::ceil((1.0 - ymin) * 0.5 * H - 0.5) + 1);
    }
    if (x1 < x0 || y1 < y0) return false;
    rect[0] = x0; rect[1] = y0; rect[2] = x1 - x0 + 1; rect[3] = y1 - y0 + 1;
    return true;
}

// Screen rectangle (view pixels, clipped) that holds every pixel whose ray can meet brick b.
// Returns false if the brick is outside the frustum.
bool brick_rect(const vr_ctx* ctx, int bid, int rect[4]) {
    const CubeDesc& c = ctx->cube;
    int b[3] = {bid % c.G[0], (bid / c.G[0]) % c.G[1], bid / (c.G[0] * c.G[1])};
    double lo[3], hi[3];
    for (int a = 0; a < 3; ++a) {
        lo[a] = (double)b[a] * c.B[a];
        hi[a] = std::min((double)(b[a] + 1) * c.B[a], (double)(c.N[a] - 1));
        if (hi[a] < lo[a]) return false;
    }
    Corner k[8];
    const Corner* kp[8];
    for (int i = 0; i < 8; ++i) {
        k[i] = project_corner(ctx->M, (i & 1) ? hi[0] : lo[0], (i & 2) ? hi[1] : lo[1], (i & 4) ? hi[2] : lo[2]);
        kp[i] = &k[i];
    }
    return rect_of_corners(ctx->view.W, ctx->view.H, kp, rect);
}

// The same rectangles for many bricks of one view: neighbouring bricks share their corners (the upper face of brick b
// is the lower face of brick b + 1, the last brick ends at N - 1), so the (G0+1)(G1+1)(G2+1) grid corners are projected
// once (vr_render_sortlast: 1024 bricks of a C4 panel cost 8192 projections per call, 25 calls per frame).
void project_corner_grid(const vr_ctx* ctx, std::vector<Corner>& grid) {
    const CubeDesc& c = ctx->cube;
    const int n0 = c.G[0] + 1, n1 = c.G[1] + 1, n2 = c.G[2] + 1;
    grid.resize((size_t)n0 * n1 * n2);
    auto at = [&](int a, int i) { return i < c.G[a] ? (double)i * c.B[a] : (double)(c.N[a] - 1); };   // = lo of brick i = hi of brick i - 1
    size_t e = 0;
    for (int iz = 0; iz < n2; ++iz)
        for (int iy = 0; iy < n1; ++iy)
            for (int ix = 0; ix < n0; ++ix) grid[e++] = project_corner(ctx->M, at(0, ix), at(1, iy), at(2, iz));
}

bool brick_rect_grid(const vr_ctx* ctx, const std::vector<Corner>& grid, int bid, int rect[4]) {
    const CubeDesc& c = ctx->cube;
    const int n0 = c.G[0] + 1, n1 = c.G[1] + 1;
    const int b[3] = {bid % c.G[0], (bid / c.G[0]) % c.G[1], bid / (c.G[0] * c.G[1])};
    const Corner* kp[8];
    for (int i = 0; i < 8; ++i)
        kp[i] = &grid[(size_t)(b[0] + (i & 1)) + (size_t)n0 * ((b[1] + ((i >> 1) & 1)) + (size_t)n1 * (b[2] + ((i >> 2) & 1)))];
    return rect_of_corners(ctx->view.W, ctx->view.H, kp, rect);
}

// A context is bound to one device: make it current for the calling thread (a process may drive several GPUs).
void enter(const vr_ctx* ctx) {
    int cur = -1;
    if (cudaGetDevice(&cur) != cudaSuccess || cur != ctx->device) cudaSetDevice(ctx->device);
}

int check_render_state(vr_ctx* ctx, bool need_tf) {
    if (!ctx) return VR_ERR_INVALID_ARG;
    enter(ctx);
    if (!ctx->has_cube) return fail(ctx, VR_ERR_STATE, "no cube: call vr_upload_cube / vr_generate_cube first");
    if (!ctx->has_view) return fail(ctx, VR_ERR_STATE, "no view: call vr_set_view first");
    if (need_tf && !ctx->has_tf) return fail(ctx, VR_ERR_STATE, "no transfer function: call vr_set_transfer_function first");
    return VR_OK;
}

// Per-brick partial images by maximum intensity in object order (vr_mip_tiles.cu: the bricks' tiles stream through
// shared memory); float32 voxels on the micro-block layout.
bool use_mip_tiles(const vr_ctx* ctx, int mode) {
    if (mode != VR_MODE_MIP || ctx->cube.layout != 1 || ctx->cube.vtype != 0 || ctx->opt_mip_tiles == 0) return false;
    // measured on C3 (64 GiB, rays 3.5 - 7 voxels apart): 30.7 ms per frame against 14.7 ms of the image-order lockstep
    // marcher: on request only
    return ctx->opt_mip_tiles > 0;
}

// Object-tile prefix of the descriptors (PartialDev::otile0); returns the total.
int number_object_tiles(const vr_ctx* ctx, PartialDev* v, int n) {
    int total = 0;
    for (int i = 0; i < n; ++i) { v[i].otile0 = total; total += object_tiles_of_brick(ctx->cube, v[i].b); }
    return total;
}

int ensure_rays(vr_ctx* ctx, int slot) {
    const size_t need = ray_buffer_bytes(ctx->view.W, ctx->view.H);
    if (ctx->rays_bytes[slot] >= need) return VR_OK;
    if (ctx->d_rays[slot]) { VR_CUDA(ctx, cudaDeviceSynchronize()); cudaFree(ctx->d_rays[slot]); }
    ctx->d_rays[slot] = nullptr; ctx->rays_bytes[slot] = 0;
    VR_CUDA(ctx, cudaMalloc(&ctx->d_rays[slot], need));
    ctx->rays_bytes[slot] = need;
    return VR_OK;
}

int upload_partials(vr_ctx* ctx, int mode, const vr_partial* hp, int n, bool with_tiles, int* total_tiles, cudaStream_t s, int* object_tiles = nullptr) {
    if (n > (int)ctx->partials_cap) {
        if (ctx->d_partials) cudaFree(ctx->d_partials);
        ctx->d_partials = nullptr;
        size_t cap = std::max<size_t>(256, (size_t)n * 2);
        VR_CUDA(ctx, cudaMalloc(&ctx->d_partials, cap * sizeof(PartialDev)));
        ctx->partials_cap = cap;
    }
    std::vector<PartialDev> v(n);
    int tiles = 0;
    const int W = ctx->view.W, H = ctx->view.H;
    for (int i = 0; i < n; ++i) {
        const vr_partial& p = hp[i];
        // the brick id is used by the marchers only (with_tiles); the compositor folds images whatever they show
        if ((with_tiles && (p.brick < ctx->cube.win_lo || p.brick >= ctx->cube.win_hi)) || p.w <= 0 || p.h <= 0 || p.x0 < 0 || p.y0 < 0 ||
            p.x0 + p.w > W || p.y0 + p.h > H || !p.d_data || p.pitch_px < (size_t)p.w)
            return fail(ctx, VR_ERR_INVALID_ARG, "bad vr_partial entry");
        if (((uintptr_t)p.d_data & (mode == VR_MODE_EA ? 15 : 3)) != 0)
            return fail(ctx, VR_ERR_INVALID_ARG, "vr_partial.d_data misaligned");
        set_brick(v[i], ctx->cube, p.brick); v[i].x0 = p.x0; v[i].y0 = p.y0; v[i].w = p.w; v[i].h = p.h;
        v[i].pitch = (long long)p.pitch_px; v[i].data = p.d_data; v[i].tile0 = tiles;
        if (with_tiles) tiles += ((p.w + kTileW - 1) / kTileW) * ((p.h + kTileH - 1) / kTileH);
    }
    if (total_tiles) *total_tiles = tiles;
    if (object_tiles) *object_tiles = number_object_tiles(ctx, v.data(), n);
    if (n > 0) VR_CUDA(ctx, cudaMemcpyAsync(ctx->d_partials, v.data(), sizeof(PartialDev) * n, cudaMemcpyHostToDevice, s));
    return VR_OK;
}

}  // namespace

namespace vr {

size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

void fill_cube_desc(CubeDesc& c, int nx, int ny, int nz, int bx, int by, int bz, int layout, int vtype) {
    std::memset(&c, 0, sizeof(c));
    c.layout = layout;
    c.vtype = vtype;
    int N[3] = {nx, ny, nz}, B[3] = {bx, by, bz};
    for (int a = 0; a < 3; ++a) {
        c.N[a] = N[a]; c.B[a] = std::min(B[a], N[a]);
        c.G[a] = (c.N[a] + c.B[a] - 1) / c.B[a];
        c.P[a] = c.B[a] + 1;
        c.sh[a] = -1;
        for (int s = 0; s < 30; ++s) if ((1 << s) == c.B[a]) c.sh[a] = s;
        c.C[a] = (c.B[a] + kCell - 1) / kCell;
    }
    if (layout == 0) c.P[0] = (c.P[0] + 3) / 4 * 4;
    c.T[0] = (c.P[0] + 3) / 4; c.T[1] = (c.P[1] + 3) / 4; c.T[2] = (c.P[2] + 1) / 2;
    c.nbricks = c.G[0] * c.G[1] * c.G[2];
    c.win_lo = 0; c.win_hi = c.nbricks;
    c.cells_per_brick = c.C[0] * c.C[1] * c.C[2];
    c.cell_words_per_brick = (c.cells_per_brick + 31) / 32;
    c.occ_words_per_brick = c.T[0] * c.T[1] * c.T[2];
    c.stride = layout == 0 ? (long long)align_up((size_t)c.P[0] * c.P[1] * c.P[2], 32)
                           : 32LL * c.T[0] * c.T[1] * c.T[2];
}

size_t cube_bytes(const CubeDesc& c) { return (size_t)(c.win_hi - c.win_lo) * (size_t)c.stride * (c.vtype == 1 ? 2 : sizeof(float)); }

MetaLayout meta_layout(const CubeDesc& c) {
    MetaLayout m;
    const size_t nb = (size_t)(c.win_hi - c.win_lo);
    size_t off = 0;
    m.brick_mm = off; off = align_up(off + sizeof(float2) * nb, 256);
    m.cell_mm = off; off = align_up(off + sizeof(float2) * nb * c.cells_per_brick, 256);
    m.cell_bits = off; off = align_up(off + sizeof(unsigned) * nb * c.cell_words_per_brick, 256);
    m.brick_active = off; off = align_up(off + sizeof(int) * nb, 256);
    m.occ = off; off = align_up(off + sizeof(unsigned) * nb * c.occ_words_per_brick, 256);
    m.hot = off; off = align_up(off + sizeof(unsigned) * nb * c.occ_words_per_brick, 256);
    m.total = off;
    return m;
}

}  // namespace vr

extern "C" {

const char* vr_status_string(int status) {
    switch (status) {
        case VR_OK: return "VR_OK";
        case VR_ERR_INVALID_ARG: return "VR_ERR_INVALID_ARG";
        case VR_ERR_BUFFER: return "VR_ERR_BUFFER";
        case VR_ERR_CUDA: return "VR_ERR_CUDA";
        case VR_ERR_STATE: return "VR_ERR_STATE";
        case VR_ERR_UNSUPPORTED: return "VR_ERR_UNSUPPORTED";
        default: return "VR_ERR_UNKNOWN";
    }
}

const char* vr_last_error(const vr_ctx* ctx) { return ctx ? ctx->err.c_str() : "null context"; }

int vr_create(vr_ctx** out, int device) {
    if (!out) return VR_ERR_INVALID_ARG;
    *out = nullptr;
    int n = 0;
    if (cudaGetDeviceCount(&n) != cudaSuccess || device < 0 || device >= n) return VR_ERR_CUDA;
    vr_ctx* ctx = new vr_ctx();
    ctx->device = device;
    cudaError_t e = cudaSetDevice(device);
    if (e == cudaSuccess) e = cudaMalloc(&ctx->d_tf_baked, 256 * sizeof(float4));
    if (e == cudaSuccess) e = cudaMalloc(&ctx->d_tf_raw, 256 * sizeof(float4));
    if (e == cudaSuccess) e = cudaMalloc(&ctx->d_counters, kNumCounters * sizeof(unsigned long long));
    if (e == cudaSuccess) e = cudaMemset(ctx->d_counters, 0, kNumCounters * sizeof(unsigned long long));
    if (e == cudaSuccess) e = cudaMalloc(&ctx->d_scratch, 8 * sizeof(unsigned long long));
    if (e != cudaSuccess) { vr_destroy(ctx); return VR_ERR_CUDA; }
    *out = ctx;
    return VR_OK;
}

int vr_destroy(vr_ctx* ctx) {
    if (!ctx) return VR_ERR_INVALID_ARG;
    cudaSetDevice(ctx->device);
    if (ctx->d_tf_baked) cudaFree(ctx->d_tf_baked);
    if (ctx->d_tf_raw) cudaFree(ctx->d_tf_raw);
    if (ctx->d_counters) cudaFree(ctx->d_counters);
    if (ctx->d_scratch) cudaFree(ctx->d_scratch);
    if (ctx->d_partials) cudaFree(ctx->d_partials);
    for (float4* r : ctx->d_rays) if (r) cudaFree(r);
    for (void* b : ctx->ipc_bases) cudaIpcCloseMemHandle(b);
    if (ctx->h_pin) cudaFreeHost(ctx->h_pin);
    if (ctx->d_pin) cudaFree(ctx->d_pin);
    for (cudaEvent_t e : ctx->pin_done) if (e) cudaEventDestroy(e);
    delete ctx;
    return VR_OK;
}

int vr_cube_layout(int nx, int ny, int nz, int bx, int by, int bz, size_t* cube_bytes_out, size_t* meta_bytes_out) {
    if (!valid_dims(nx, ny, nz, bx, by, bz) || !cube_bytes_out || !meta_bytes_out) return VR_ERR_INVALID_ARG;
    CubeDesc c0, c1;                       // enough for either in-brick layout (VR_OPT_LAYOUT)
    fill_cube_desc(c0, nx, ny, nz, bx, by, bz, 0);
    fill_cube_desc(c1, nx, ny, nz, bx, by, bz, 1);
    *cube_bytes_out = std::max(cube_bytes(c0), cube_bytes(c1));
    *meta_bytes_out = std::max(meta_layout(c0).total, meta_layout(c1).total);
    return VR_OK;
}

int vr_cube_layout_typed(int nx, int ny, int nz, int bx, int by, int bz, int voxel_type, int first_brick, int end_brick,
                         size_t* cube_bytes_out, size_t* meta_bytes_out) {
    if (!valid_dims(nx, ny, nz, bx, by, bz) || !cube_bytes_out || !meta_bytes_out || (voxel_type != 0 && voxel_type != 1)) return VR_ERR_INVALID_ARG;
    CubeDesc c;
    fill_cube_desc(c, nx, ny, nz, bx, by, bz, 1, voxel_type);
    if (end_brick >= 0) {
        if (first_brick < 0 || end_brick < first_brick || end_brick > c.nbricks) return VR_ERR_INVALID_ARG;
        c.win_lo = first_brick; c.win_hi = end_brick;
    }
    *cube_bytes_out = std::max<size_t>(256, cube_bytes(c));
    *meta_bytes_out = std::max<size_t>(256, meta_layout(c).total);
    return VR_OK;
}

int vr_meta_static_bytes(int nx, int ny, int nz, int bx, int by, int bz, int voxel_type, int first_brick, int end_brick,
                         size_t* static_bytes_out) {
    if (!valid_dims(nx, ny, nz, bx, by, bz) || !static_bytes_out || (voxel_type != 0 && voxel_type != 1)) return VR_ERR_INVALID_ARG;
    CubeDesc c;
    fill_cube_desc(c, nx, ny, nz, bx, by, bz, 1, voxel_type);
    if (end_brick >= 0) {
        if (first_brick < 0 || end_brick < first_brick || end_brick > c.nbricks) return VR_ERR_INVALID_ARG;
        c.win_lo = first_brick; c.win_hi = end_brick;
    }
    *static_bytes_out = meta_layout(c).cell_bits;           // (min,max) per brick and per macro-cell lead the meta buffer
    return VR_OK;
}

int vr_attach_cube(vr_ctx* ctx, int nx, int ny, int nz, int bx, int by, int bz, const void* d_cube, void* d_meta) {
    VR_RANGE();
    if (!ctx) return VR_ERR_INVALID_ARG;
    enter(ctx);
    if (!valid_dims(nx, ny, nz, bx, by, bz) || !d_cube || !d_meta) return fail(ctx, VR_ERR_INVALID_ARG, "vr_attach_cube: bad argument");
    fill_cube_desc(ctx->cube, nx, ny, nz, bx, by, bz, ctx->opt_layout, ctx->opt_vtype);
    apply_window(ctx, ctx->cube);
    bind_meta(ctx->cube, d_cube, d_meta);
    int rc = fetch_brick_mm(ctx, nullptr);
    if (rc) return rc;
    ctx->has_cube = true;
    ctx->activity_dirty = true; ctx->key_valid = false; ctx->occ_valid = false;
    return VR_OK;
}

int vr_upload_cube(vr_ctx* ctx, const float* src, int src_is_device, int nx, int ny, int nz, int bx, int by,
                   int bz, void* d_cube, void* d_meta, void* stream) {
    VR_RANGE();
    if (!ctx) return VR_ERR_INVALID_ARG;
    enter(ctx);
    if (!valid_dims(nx, ny, nz, bx, by, bz) || !src || !d_cube || !d_meta) return fail(ctx, VR_ERR_INVALID_ARG, "vr_upload_cube: bad argument");
    cudaStream_t s = (cudaStream_t)stream;
    ctx->has_cube = false;
    CubeDesc& c = ctx->cube;
    fill_cube_desc(c, nx, ny, nz, bx, by, bz, ctx->opt_layout, ctx->opt_vtype);
    apply_window(ctx, c);
    bind_meta(c, d_cube, d_meta);
    VR_CUDA(ctx, cudaMemsetAsync(d_cube, 0, cube_bytes(c), s));
    VR_CUDA(ctx, cudaMemsetAsync(ctx->d_scratch, 0, sizeof(unsigned long long), s));
    if (src_is_device) {
        VR_CUDA(ctx, launch_rebrick(c, const_cast<float*>(c.cube), src, 0, nz, ctx->d_scratch, s));
        ctx->launches += 1;
    } else {
        // two staging slabs of whole planes (about 128 MiB each): the copy of slab i + 1 (internal copy
        // stream) overlaps the rebricking of slab i (caller's stream); freed again before returning
        const size_t plane = (size_t)nx * ny * sizeof(float);
        const int planes = (int)std::max<size_t>(1, std::min<size_t>((size_t)nz, ((size_t)128 << 20) / plane));
        const size_t slab = plane * planes;
        float* stage[2] = {nullptr, nullptr};
        cudaStream_t cs = nullptr;
        cudaEvent_t copied[2] = {nullptr, nullptr}, freed[2] = {nullptr, nullptr};
        cudaError_t e = cudaStreamCreateWithFlags(&cs, cudaStreamNonBlocking);
        for (int i = 0; i < 2 && e == cudaSuccess; ++i) {
            e = cudaMalloc(&stage[i], slab);
            if (e == cudaSuccess) e = cudaEventCreateWithFlags(&copied[i], cudaEventDisableTiming);
            if (e == cudaSuccess) e = cudaEventCreateWithFlags(&freed[i], cudaEventDisableTiming);
        }
        int i = 0;
        for (int z0 = 0; z0 < nz && e == cudaSuccess; z0 += planes, ++i) {
            const int z1 = std::min(nz, z0 + planes), bsel = i & 1;
            if (i >= 2) e = cudaStreamWaitEvent(cs, freed[bsel], 0);               // the slab's previous content was rebricked
            if (e == cudaSuccess) e = cudaMemcpyAsync(stage[bsel], src + (size_t)z0 * nx * ny, plane * (z1 - z0), cudaMemcpyHostToDevice, cs);
            if (e == cudaSuccess) e = cudaEventRecord(copied[bsel], cs);
            if (e == cudaSuccess) e = cudaStreamWaitEvent(s, copied[bsel], 0);
            if (e == cudaSuccess) e = launch_rebrick(c, const_cast<float*>(c.cube), stage[bsel], z0, z1, ctx->d_scratch, s);
            if (e == cudaSuccess) e = cudaEventRecord(freed[bsel], s);
            ctx->launches += 1;
        }
        if (e == cudaSuccess) e = cudaStreamSynchronize(s);
        for (int k = 0; k < 2; ++k) {
            if (stage[k]) cudaFree(stage[k]);
            if (copied[k]) cudaEventDestroy(copied[k]);
            if (freed[k]) cudaEventDestroy(freed[k]);
        }
        if (cs) cudaStreamDestroy(cs);
        if (e != cudaSuccess) return cuda_fail(ctx, e, "vr_upload_cube (host source)");
    }
    unsigned long long n_bad = 0;
    VR_CUDA(ctx, cudaMemcpyAsync(&n_bad, ctx->d_scratch, sizeof(n_bad), cudaMemcpyDeviceToHost, s));
    VR_CUDA(ctx, cudaStreamSynchronize(s));
    if (n_bad) return fail(ctx, VR_ERR_INVALID_ARG, "vr_upload_cube: the cube holds " + std::to_string(n_bad) + " non-finite voxels (NaN / inf)");
    return finish_cube(ctx, s);
}

int vr_generate_cube(vr_ctx* ctx, const vr_gen_params* prm, uint64_t seed, int nx, int ny, int nz, int bx,
                     int by, int bz, void* d_cube, void* d_meta, void* stream) {
    VR_RANGE();
    if (!ctx) return VR_ERR_INVALID_ARG;
    enter(ctx);
    if (!valid_dims(nx, ny, nz, bx, by, bz) || !prm || !d_cube || !d_meta) return fail(ctx, VR_ERR_INVALID_ARG, "vr_generate_cube: bad argument");
    if (prm->n_sources < 0 || prm->n_zero_boxes < 0 || (prm->n_sources > 0 && !prm->h_sources) ||
        (prm->n_zero_boxes > 0 && !prm->h_zero_boxes))
        return fail(ctx, VR_ERR_INVALID_ARG, "vr_generate_cube: bad source / zero-box list");
    cudaStream_t s = (cudaStream_t)stream;
    ctx->has_cube = false;
    CubeDesc& c = ctx->cube;
    fill_cube_desc(c, nx, ny, nz, bx, by, bz, ctx->opt_layout, ctx->opt_vtype);
    apply_window(ctx, c);
    bind_meta(c, d_cube, d_meta);
    // bin the sources (ascending id) and the zero boxes over 32^3 tiles of the cube
    const int T[3] = {(nx + 31) / 32, (ny + 31) / 32, (nz + 31) / 32};
    const size_t ntile = (size_t)T[0] * T[1] * T[2];
    std::vector<int> cnt(ntile + 1, 0);
    std::vector<char> zflag(ntile, 0);
    auto for_tiles = [&](const double* box, auto&& fn) {
        int lo[3], hi[3];
        const int N[3] = {nx, ny, nz};
        for (int a = 0; a < 3; ++a) {
            lo[a] = std::max(0, (int)box[2 * a]) >> 5;
            hi[a] = std::min(N[a] - 1, (int)box[2 * a + 1]) >> 5;
        }
        for (int z = lo[2]; z <= hi[2]; ++z) for (int y = lo[1]; y <= hi[1]; ++y) for (int x = lo[0]; x <= hi[0]; ++x)
            fn((size_t)x + T[0] * ((size_t)y + (size_t)T[1] * z));
    };
    for (int i = 0; i < prm->n_sources; ++i) for_tiles(prm->h_sources + 16 * (size_t)i + 10, [&](size_t t) { cnt[t + 1]++; });
    for (size_t t = 0; t < ntile; ++t) cnt[t + 1] += cnt[t];
    std::vector<int> ids((size_t)cnt[ntile] + 1), fillp(cnt.begin(), cnt.end() - 1);
    for (int i = 0; i < prm->n_sources; ++i) for_tiles(prm->h_sources + 16 * (size_t)i + 10, [&](size_t t) { ids[fillp[t]++] = i; });
    for (int i = 0; i < prm->n_zero_boxes; ++i) {
        double box[6];
        for (int k = 0; k < 6; ++k) box[k] = prm->h_zero_boxes[6 * i + k];
        for_tiles(box, [&](size_t t) { zflag[t] = 1; });
    }
    std::vector<int> offs(cnt);
    for (size_t t = 0; t < ntile; ++t) if (zflag[t]) offs[t] = ~offs[t];
    double* d_src = nullptr; int* d_offs = nullptr; int* d_ids = nullptr; int* d_zb = nullptr;
    auto cleanup = [&]() { cudaFree(d_src); cudaFree(d_offs); cudaFree(d_ids); cudaFree(d_zb); };
    cudaError_t e = cudaMalloc(&d_src, sizeof(double) * 16 * std::max(1, prm->n_sources));
    if (e == cudaSuccess) e = cudaMalloc(&d_offs, sizeof(int) * offs.size());
    if (e == cudaSuccess) e = cudaMalloc(&d_ids, sizeof(int) * ids.size());
    if (e == cudaSuccess) e = cudaMalloc(&d_zb, sizeof(int) * 6 * std::max(1, prm->n_zero_boxes));
    if (e == cudaSuccess && prm->n_sources) e = cudaMemcpyAsync(d_src, prm->h_sources, sizeof(double) * 16 * prm->n_sources, cudaMemcpyHostToDevice, s);
    if (e == cudaSuccess) e = cudaMemcpyAsync(d_offs, offs.data(), sizeof(int) * offs.size(), cudaMemcpyHostToDevice, s);
    if (e == cudaSuccess) e = cudaMemcpyAsync(d_ids, ids.data(), sizeof(int) * ids.size(), cudaMemcpyHostToDevice, s);
    if (e == cudaSuccess && prm->n_zero_boxes) e = cudaMemcpyAsync(d_zb, prm->h_zero_boxes, sizeof(int) * 6 * prm->n_zero_boxes, cudaMemcpyHostToDevice, s);
    if (e == cudaSuccess) {
        GenDev g;
        g.sources = d_src; g.tile_offsets = d_offs; g.tile_ids = d_ids;
        g.tiles[0] = T[0]; g.tiles[1] = T[1]; g.tiles[2] = T[2];
        g.zero_boxes = d_zb; g.n_zero = prm->n_zero_boxes; g.continuum = prm->continuum; g.seed = seed;
        e = launch_generate(c, const_cast<float*>(c.cube), g, s);
        ctx->launches += 1;
    }
    if (e == cudaSuccess) e = cudaStreamSynchronize(s);
    cleanup();
    if (e != cudaSuccess) return cuda_fail(ctx, e, "vr_generate_cube");
    return finish_cube(ctx, s);
}

int vr_download_brick(vr_ctx* ctx, int brick_id, float* d_dst, void* stream) {
    VR_RANGE();
    if (!ctx) return VR_ERR_INVALID_ARG;
    enter(ctx);
    if (!ctx->has_cube) return fail(ctx, VR_ERR_STATE, "no cube");
    if (brick_id < ctx->cube.win_lo || brick_id >= ctx->cube.win_hi || !d_dst) return fail(ctx, VR_ERR_INVALID_ARG, "vr_download_brick: bad argument (brick not resident?)");
    VR_CUDA(ctx, launch_unbrick(ctx->cube, brick_id, d_dst, (cudaStream_t)stream));
    ctx->launches += 1;
    return VR_OK;
}

int vr_set_view(vr_ctx* ctx, const float mvp[16], int width, int height, float step) {
    VR_RANGE();
    if (!ctx) return VR_ERR_INVALID_ARG;
    if (!mvp || width <= 0 || height <= 0 || !(step > 0.f) || !std::isfinite(step)) return fail(ctx, VR_ERR_INVALID_ARG, "vr_set_view: bad argument");
    double M[16], Minv[16];
    for (int i = 0; i < 16; ++i) { M[i] = (double)mvp[i]; if (!std::isfinite(M[i])) return fail(ctx, VR_ERR_INVALID_ARG, "vr_set_view: non-finite matrix"); }
    if (!invert4(M, Minv)) return fail(ctx, VR_ERR_INVALID_ARG, "vr_set_view: singular matrix");
    std::memcpy(ctx->M, M, sizeof(M)); std::memcpy(ctx->Minv, Minv, sizeof(Minv));
    std::memcpy(ctx->view.Minv, Minv, sizeof(Minv));
    ctx->view.W = width; ctx->view.H = height; ctx->view.step = step;
    ctx->view.vx0 = 0; ctx->view.vy0 = 0; ctx->view.pitch = width;
    ctx->has_view = true;
    return VR_OK;
}

int vr_set_viewport(vr_ctx* ctx, int x0, int y0, size_t pitch_px) {
    if (!ctx) return VR_ERR_INVALID_ARG;
    if (!ctx->has_view) return fail(ctx, VR_ERR_STATE, "vr_set_viewport before vr_set_view");
    if (x0 < 0 || y0 < 0 || pitch_px < (size_t)(x0 + ctx->view.W)) return fail(ctx, VR_ERR_INVALID_ARG, "vr_set_viewport: bad argument");
    ctx->view.vx0 = x0; ctx->view.vy0 = y0; ctx->view.pitch = (long long)pitch_px;
    return VR_OK;
}

int vr_set_transfer_function(vr_ctx* ctx, const float rgba[1024], float vmin, float vmax) {
    VR_RANGE();
    if (!ctx) return VR_ERR_INVALID_ARG;
    if (!rgba || !(vmax > vmin) || !std::isfinite(vmin) || !std::isfinite(vmax)) return fail(ctx, VR_ERR_INVALID_ARG, "vr_set_transfer_function: bad argument");
    for (int i = 0; i < 1024; ++i) if (!(rgba[i] >= 0.f && rgba[i] <= 1.f)) return fail(ctx, VR_ERR_INVALID_ARG, "vr_set_transfer_function: entries must lie in [0,1]");
    std::memcpy(ctx->tf_raw, rgba, sizeof(ctx->tf_raw));
    ctx->vmin = vmin; ctx->vmax = vmax;
    ctx->scale = (float)(255.0 / ((double)vmax - (double)vmin));
    ctx->has_tf = true; ctx->tables_dirty = true;
    return VR_OK;
}

int vr_render_mip(vr_ctx* ctx, float* d_out, float* d_out_rgba, float miss, void* stream) {
    VR_RANGE();
    int rc = check_render_state(ctx, d_out_rgba != nullptr);
    if (rc) return rc;
    if (!d_out) return fail(ctx, VR_ERR_INVALID_ARG, "vr_render_mip: null output");
    if (ctx->cube.win_hi - ctx->cube.win_lo != ctx->cube.nbricks) return fail(ctx, VR_ERR_STATE, "vr_render_mip needs the whole cube resident (brick window set: use vr_render_bricks)");
    cudaStream_t s = (cudaStream_t)stream;
    if ((rc = ensure_tables(ctx, s))) return rc;
    RenderArgs a{};
    a.mode = VR_MODE_MIP; a.tau = 2.f; a.miss = miss; a.skip = skip_level(ctx, a.mode); a.variant = pick_variant(ctx, a.mode, a.skip); a.ring = resolve_ring(ctx, a.mode);
    a.out = d_out; a.out_rgba = d_out_rgba; a.counters = ctx->d_counters;
    VR_CUDA(ctx, launch_render_global(ctx->cube, ctx->view, tf_desc(ctx), a, s));
    ctx->launches += 1;
    return VR_OK;
}

int vr_render_ea(vr_ctx* ctx, float* d_out, const float bg[4], float tau, void* stream) {
    VR_RANGE();
    int rc = check_render_state(ctx, true);
    if (rc) return rc;
    if (!d_out || !bg || !(tau > 0.f)) return fail(ctx, VR_ERR_INVALID_ARG, "vr_render_ea: bad argument");
    if (((uintptr_t)d_out & 15) != 0) return fail(ctx, VR_ERR_INVALID_ARG, "vr_render_ea: output must be 16-byte aligned");
    if (ctx->cube.win_hi - ctx->cube.win_lo != ctx->cube.nbricks) return fail(ctx, VR_ERR_STATE, "vr_render_ea needs the whole cube resident (brick window set: use vr_render_bricks)");
    cudaStream_t s = (cudaStream_t)stream;
    if ((rc = ensure_tables(ctx, s))) return rc;
    RenderArgs a{};
    a.mode = VR_MODE_EA; a.tau = tau; a.skip = skip_level(ctx, a.mode); a.variant = pick_variant(ctx, a.mode, a.skip); a.dense = resolve_dense(ctx); a.ring = resolve_ring(ctx, a.mode);
    for (int i = 0; i < 4; ++i) a.bg[i] = bg[i];
    a.out = d_out; a.counters = ctx->d_counters;
    if ((rc = ensure_occ(ctx, a.skip, s))) return rc;
    VR_CUDA(ctx, launch_render_global(ctx->cube, ctx->view, tf_desc(ctx), a, s));
    ctx->launches += 1;
    return VR_OK;
}

// O-9 visibility key of every brick under the current view: perspective, eye = h.xyz / h.w with
// h = Minv (0,0,1,0)^T, key = sum |b_a - E_a|; orthographic: b_a counted along the common direction.
static void brick_keys(const vr_ctx* ctx, std::vector<int>& key) {
    const CubeDesc& c = ctx->cube;
    const double* Mi = ctx->Minv;
    double h[4] = {Mi[2], Mi[6], Mi[10], Mi[14]};
    double nrm = std::fabs(h[0]) + std::fabs(h[1]) + std::fabs(h[2]);
    double nmax = (double)std::max(c.N[0], std::max(c.N[1], c.N[2]));
    bool persp = std::fabs(h[3]) * nmax * 1e9 > nrm;
    int E[3] = {0, 0, 0}, sg[3] = {0, 0, 0};
    if (persp) {
        // an eye far outside the grid: any index beyond the grid's ends gives the same order (every |b_a - E_a|
        // moves by one constant), so clamp before the int cast
        for (int a = 0; a < 3; ++a) E[a] = (int)std::min((double)c.G[a], std::max(-1.0, std::floor((h[a] / h[3]) / (double)c.B[a])));
    } else {
        // direction of the central ray: far point minus near point
        double pn[4], pf[4];
        for (int r = 0; r < 4; ++r) { pn[r] = -Mi[4 * r + 2] + Mi[4 * r + 3]; pf[r] = Mi[4 * r + 2] + Mi[4 * r + 3]; }
        double L = 0, d[3];
        for (int a = 0; a < 3; ++a) { d[a] = pf[a] / pf[3] - pn[a] / pn[3]; L += d[a] * d[a]; }
        L = std::sqrt(L);
        for (int a = 0; a < 3; ++a) sg[a] = d[a] / L > 1e-12 ? 1 : (d[a] / L < -1e-12 ? -1 : 0);
    }
    key.resize(c.nbricks);
    for (int bid = 0; bid < c.nbricks; ++bid) {
        int b[3] = {bid % c.G[0], (bid / c.G[0]) % c.G[1], bid / (c.G[0] * c.G[1])};
        int k = 0;
        for (int a = 0; a < 3; ++a)
            k += persp ? std::abs(b[a] - E[a]) : (sg[a] > 0 ? b[a] : (sg[a] < 0 ? c.G[a] - 1 - b[a] : 0));
        key[bid] = k;
    }
}

int vr_sort_bricks(vr_ctx* ctx, int mode, int* h_order, int* n_active) {
    VR_RANGE();
    int rc = check_render_state(ctx, mode == VR_MODE_EA);
    if (rc) return rc;
    if (!n_active || (mode != VR_MODE_MIP && mode != VR_MODE_EA)) return fail(ctx, VR_ERR_INVALID_ARG, "vr_sort_bricks: bad argument");
    const CubeDesc& c = ctx->cube;
    if (mode == VR_MODE_EA && (ctx->tables_dirty || ctx->baked_step != ctx->view.step)) { bake_tf(ctx); ctx->tables_dirty = true; }
    std::vector<int> key;
    brick_keys(ctx, key);
    std::vector<std::pair<int, int>> keyed;
    keyed.reserve(c.win_hi - c.win_lo);
    for (int bid = c.win_lo; bid < c.win_hi; ++bid) {      // resident bricks only
        int rect[4];
        if (!brick_rect(ctx, bid, rect)) continue;
        if (mode == VR_MODE_EA && ctx->opt_skip && !range_active(ctx, ctx->h_brick_mm[bid].x, ctx->h_brick_mm[bid].y)) continue;
        keyed.emplace_back(key[bid], bid);
    }
    std::stable_sort(keyed.begin(), keyed.end());
    *n_active = (int)keyed.size();
    if (h_order) for (size_t i = 0; i < keyed.size(); ++i) h_order[i] = keyed[i].second;
    return VR_OK;
}

int vr_sort_groups(vr_ctx* ctx, const int* h_group_first, int n_groups, int* h_group_order) {
    VR_RANGE();
    int rc = check_render_state(ctx, false);
    if (rc) return rc;
    if (!h_group_first || !h_group_order || n_groups <= 0) return fail(ctx, VR_ERR_INVALID_ARG, "vr_sort_groups: bad argument");
    const CubeDesc& c = ctx->cube;
    const int layer = c.G[0] * c.G[1];
    for (int g = 0; g <= n_groups; ++g) {
        const int f = h_group_first[g];
        if (f < 0 || f > c.nbricks || f % layer != 0 || (g > 0 && f < h_group_first[g - 1]))
            return fail(ctx, VR_ERR_INVALID_ARG, "vr_sort_groups: groups must be ascending whole z-layers of bricks");
    }
    if (h_group_first[0] != 0 || h_group_first[n_groups] != c.nbricks)
        return fail(ctx, VR_ERR_INVALID_ARG, "vr_sort_groups: groups must cover all bricks");
    std::vector<int> key;
    brick_keys(ctx, key);
    std::vector<std::pair<int, int>> keyed;
    for (int g = 0; g < n_groups; ++g) {
        int k = INT_MAX;
        for (int bid = h_group_first[g]; bid < h_group_first[g + 1]; ++bid) k = std::min(k, key[bid]);
        keyed.emplace_back(k, g);                           // an empty group sorts last; it has no partial to fold
    }
    std::stable_sort(keyed.begin(), keyed.end());
    for (int g = 0; g < n_groups; ++g) h_group_order[g] = keyed[g].second;
    return VR_OK;
}

int vr_set_brick_window(vr_ctx* ctx, int first_brick, int end_brick) {
    if (!ctx) return VR_ERR_INVALID_ARG;
    if (end_brick < 0) { ctx->win_lo = 0; ctx->win_hi = -1; return VR_OK; }
    if (first_brick < 0 || end_brick < first_brick) return fail(ctx, VR_ERR_INVALID_ARG, "vr_set_brick_window: bad window");
    ctx->win_lo = first_brick; ctx->win_hi = end_brick;
    return VR_OK;
}

int vr_window_layout(int nx, int ny, int nz, int bx, int by, int bz, int first_brick, int end_brick, size_t* cube_bytes_out,
                     size_t* meta_bytes_out) {
    if (!valid_dims(nx, ny, nz, bx, by, bz) || !cube_bytes_out || !meta_bytes_out || first_brick < 0 || end_brick < first_brick)
        return VR_ERR_INVALID_ARG;
    CubeDesc c0, c1;
    fill_cube_desc(c0, nx, ny, nz, bx, by, bz, 0);
    fill_cube_desc(c1, nx, ny, nz, bx, by, bz, 1);
    if (end_brick > c0.nbricks) return VR_ERR_INVALID_ARG;
    c0.win_lo = c1.win_lo = first_brick; c0.win_hi = c1.win_hi = end_brick;
    *cube_bytes_out = std::max<size_t>(256, std::max(cube_bytes(c0), cube_bytes(c1)));     // an empty window still gets valid buffers
    *meta_bytes_out = std::max<size_t>(256, std::max(meta_layout(c0).total, meta_layout(c1).total));
    return VR_OK;
}

int vr_partial_layout(vr_ctx* ctx, int mode, const int* ids, int n, vr_partial* hp, size_t* arena_bytes) {
    VR_RANGE();
    int rc = check_render_state(ctx, false);
    if (rc) return rc;
    if (n < 0 || (n > 0 && (!ids || !hp)) || !arena_bytes || (mode != VR_MODE_MIP && mode != VR_MODE_EA))
        return fail(ctx, VR_ERR_INVALID_ARG, "vr_partial_layout: bad argument");
    const size_t px_bytes = mode == VR_MODE_EA ? 16 : 4;
    size_t off = 0;
    for (int i = 0; i < n; ++i) {
        if (ids[i] < 0 || ids[i] >= ctx->cube.nbricks) return fail(ctx, VR_ERR_INVALID_ARG, "vr_partial_layout: bad brick id");
        int rect[4];
        if (!brick_rect(ctx, ids[i], rect)) { rect[0] = rect[1] = 0; rect[2] = rect[3] = 1; }   // off-screen: 1 px
        hp[i].brick = ids[i];
        hp[i].x0 = rect[0]; hp[i].y0 = rect[1]; hp[i].w = rect[2]; hp[i].h = rect[3];
        hp[i].pitch_px = (size_t)rect[2];
        hp[i].d_data = (void*)off;
        off = align_up(off + px_bytes * (size_t)rect[2] * rect[3], 256);
    }
    *arena_bytes = off;
    return VR_OK;
}

int vr_render_bricks(vr_ctx* ctx, int mode, const vr_partial* hp, int n, float tau, void* stream) {
    VR_RANGE();
    int rc = check_render_state(ctx, mode == VR_MODE_EA);
    if (rc) return rc;
    if (n < 0 || (n > 0 && !hp) || (mode != VR_MODE_MIP && mode != VR_MODE_EA) || !(tau > 0.f))
        return fail(ctx, VR_ERR_INVALID_ARG, "vr_render_bricks: bad argument");
    cudaStream_t s = (cudaStream_t)stream;
    if ((rc = ensure_tables(ctx, s))) return rc;
    int tiles = 0, otiles = 0;
    const bool by_tiles = use_mip_tiles(ctx, mode);
    if ((rc = upload_partials(ctx, mode, hp, n, true, &tiles, s, by_tiles ? &otiles : nullptr))) return rc;
    RenderArgs a{};
    a.mode = mode; a.tau = mode == VR_MODE_EA ? tau : 2.f; a.skip = skip_level(ctx, a.mode, true); a.variant = pick_variant(ctx, a.mode, a.skip); a.dense = resolve_dense(ctx); a.ring = resolve_ring(ctx, a.mode);
    a.counters = ctx->d_counters;
    if (by_tiles) {
        if ((rc = ensure_rays(ctx, vr_ctx::kPinSlots))) return rc;
        VR_CUDA(ctx, launch_mip_tiles(ctx->cube, ctx->view, ctx->M, a, ctx->d_partials, n, tiles, otiles, ctx->d_rays[vr_ctx::kPinSlots], s));
        ctx->launches += (n > 0 && tiles > 0) ? 3 : 0;
        return VR_OK;
    }
    if ((rc = ensure_occ(ctx, a.skip, s))) return rc;
    VR_CUDA(ctx, launch_render_bricks(ctx->cube, ctx->view, tf_desc(ctx), a, ctx->d_partials, n, tiles, s));
    ctx->launches += (n > 0 && tiles > 0) ? 1 : 0;
    return VR_OK;
}

int vr_render_sortlast(vr_ctx* ctx, int mode, float tau, void* d_arena, size_t arena_bytes, size_t* needed_bytes, float* d_out,
                       const float bg[4], void* stream) {
    VR_RANGE();
    int rc = check_render_state(ctx, mode == VR_MODE_EA);
    if (rc) return rc;
    if ((mode != VR_MODE_MIP && mode != VR_MODE_EA) || !(tau > 0.f) || !d_out || !bg || !needed_bytes || (arena_bytes > 0 && !d_arena) ||
        ((uintptr_t)d_arena & 255) != 0)
        return fail(ctx, VR_ERR_INVALID_ARG, "vr_render_sortlast: bad argument (the arena must be 256-byte aligned)");
    cudaStream_t s = (cudaStream_t)stream;
    if ((rc = ensure_tables(ctx, s))) return rc;
    const CubeDesc& c = ctx->cube;
    // S1: front-to-back list of the resident bricks that can contribute, with their screen rectangles (computed once)
    brick_keys(ctx, ctx->keys);
    {   // counting sort by key, bricks of equal key in ascending id (= the stable sort of vr_sort_bricks; keys are small
        // non-negative integers, at most G0 + G1 + G2 + 3; no allocation once the scratch vectors have grown)
        int kmax = 0;
        for (int bid = c.win_lo; bid < c.win_hi; ++bid) kmax = std::max(kmax, ctx->keys[bid]);
        ctx->key_count.assign((size_t)kmax + 2, 0);
        auto live = [&](int bid) { return !(mode == VR_MODE_EA && ctx->opt_skip && !ctx->h_brick_active[bid]); };
        for (int bid = c.win_lo; bid < c.win_hi; ++bid) if (live(bid)) ++ctx->key_count[ctx->keys[bid] + 1];
        for (int k = 0; k <= kmax; ++k) ctx->key_count[k + 1] += ctx->key_count[k];
        ctx->keyed.resize((size_t)ctx->key_count[kmax + 1]);
        for (int bid = c.win_lo; bid < c.win_hi; ++bid) if (live(bid)) ctx->keyed[ctx->key_count[ctx->keys[bid]]++] = {ctx->keys[bid], bid};
    }
    project_corner_grid(ctx, ctx->corner_grid);
    // pinned slot
    const size_t cap_needed = ctx->keyed.size() + 1;
    if (ctx->pin_cap < cap_needed) {
        for (cudaEvent_t e : ctx->pin_done) if (e) cudaEventSynchronize(e);
        if (ctx->h_pin) cudaFreeHost(ctx->h_pin);
        if (ctx->d_pin) cudaFree(ctx->d_pin);
        ctx->h_pin = nullptr; ctx->d_pin = nullptr; ctx->pin_cap = 0;
        const size_t cap = std::max<size_t>(1024, 2 * cap_needed);
        VR_CUDA(ctx, cudaHostAlloc(&ctx->h_pin, sizeof(PartialDev) * cap * vr_ctx::kPinSlots, cudaHostAllocDefault));
        VR_CUDA(ctx, cudaMalloc(&ctx->d_pin, sizeof(PartialDev) * cap * vr_ctx::kPinSlots));
        ctx->pin_cap = cap;
        for (cudaEvent_t& e : ctx->pin_done) if (!e) VR_CUDA(ctx, cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
    }
    const int slot = ctx->pin_next;
    ctx->pin_next = (slot + 1) % vr_ctx::kPinSlots;
    VR_CUDA(ctx, cudaEventSynchronize(ctx->pin_done[slot]));                 // the call that last used this slot is done with it
    PartialDev* v = ctx->h_pin + (size_t)slot * ctx->pin_cap;
    PartialDev* dv = ctx->d_pin + (size_t)slot * ctx->pin_cap;
    const size_t px_bytes = mode == VR_MODE_EA ? 16 : 4;
    size_t off = 0;
    int n = 0, tiles = 0;
    for (const auto& kb : ctx->keyed) {
        int rect[4];
        if (!brick_rect_grid(ctx, ctx->corner_grid, kb.second, rect)) continue;   // outside the frustum
        PartialDev& d = v[n++];
        set_brick(d, ctx->cube, kb.second); d.x0 = rect[0]; d.y0 = rect[1]; d.w = rect[2]; d.h = rect[3]; d.tile0 = tiles;
        d.pitch = rect[2]; d.data = (char*)d_arena + off;
        tiles += ((rect[2] + kTileW - 1) / kTileW) * ((rect[3] + kTileH - 1) / kTileH);
        off = align_up(off + px_bytes * (size_t)rect[2] * rect[3], 256);
    }
    *needed_bytes = off;
    if (off > arena_bytes) return fail(ctx, VR_ERR_BUFFER, "vr_render_sortlast: the arena is too small (see *needed_bytes)");
    const bool by_tiles = use_mip_tiles(ctx, mode);
    const int otiles = by_tiles ? number_object_tiles(ctx, v, n) : 0;
    if (n > 0) VR_CUDA(ctx, cudaMemcpyAsync(dv, v, sizeof(PartialDev) * n, cudaMemcpyHostToDevice, s));
    RenderArgs a{};
    a.mode = mode; a.tau = mode == VR_MODE_EA ? tau : 2.f; a.skip = skip_level(ctx, a.mode, true); a.variant = pick_variant(ctx, a.mode, a.skip);
    a.dense = resolve_dense(ctx); a.ring = resolve_ring(ctx, a.mode);
    a.counters = ctx->d_counters;
    if (by_tiles) {
        if ((rc = ensure_rays(ctx, slot))) return rc;
        VR_CUDA(ctx, launch_mip_tiles(c, ctx->view, ctx->M, a, dv, n, tiles, otiles, ctx->d_rays[slot], s));
        ctx->launches += (n > 0 && tiles > 0) ? 2 : 0;
    } else {
        if ((rc = ensure_occ(ctx, a.skip, s))) return rc;
        VR_CUDA(ctx, launch_render_bricks(c, ctx->view, tf_desc(ctx), a, dv, n, tiles, s));
    }
    VR_CUDA(ctx, launch_composite(ctx->view, mode, dv, n, d_out, bg, s));
    VR_CUDA(ctx, cudaEventRecord(ctx->pin_done[slot], s));                   // both kernels have read the slot
    ctx->launches += (n > 0 && tiles > 0) ? 2 : 1;
    return VR_OK;
}

int vr_composite_bricks(vr_ctx* ctx, int mode, const vr_partial* hp, int n, float* d_out, const float bg[4], void* stream) {
    VR_RANGE();
    int rc = check_render_state(ctx, false);
    if (rc) return rc;
    if (n < 0 || (n > 0 && !hp) || !d_out || !bg || (mode != VR_MODE_MIP && mode != VR_MODE_EA))
        return fail(ctx, VR_ERR_INVALID_ARG, "vr_composite_bricks: bad argument");
    cudaStream_t s = (cudaStream_t)stream;
    if ((rc = upload_partials(ctx, mode, hp, n, false, nullptr, s))) return rc;
    VR_CUDA(ctx, launch_composite(ctx->view, mode, ctx->d_partials, n, d_out, bg, s));
    ctx->launches += 1;
    return VR_OK;
}

int vr_composite_bricks_static(vr_ctx* ctx, int mode, const vr_partial* hp, int n, float* d_out, const float bg[4], void* stream) {
    VR_RANGE();
    int rc = check_render_state(ctx, false);                 // makes the context's device current
    if (rc) return rc;
    if (n < 0 || (n > 0 && !hp) || !d_out || !bg || (mode != VR_MODE_MIP && mode != VR_MODE_EA))
        return fail(ctx, VR_ERR_INVALID_ARG, "vr_composite_bricks_static: bad argument");
    if (n > kStaticMaxPartials)
        return fail(ctx, VR_ERR_BUFFER, "vr_composite_bricks_static: " + std::to_string(n) + " partial images exceed the static maximum of " +
                                        std::to_string(kStaticMaxPartials) + " (VR_STATIC_MAX_PARTIALS): use vr_composite_bricks");
    cudaStream_t s = (cudaStream_t)stream;
    const int W = ctx->view.W, H = ctx->view.H;
    for (int i = 0; i < n; ++i) {                            // every entry is checked before anything is enqueued
        const vr_partial& p = hp[i];
        if (p.w <= 0 || p.h <= 0 || p.x0 < 0 || p.y0 < 0 || p.x0 + p.w > W || p.y0 + p.h > H || !p.d_data || p.pitch_px < (size_t)p.w)
            return fail(ctx, VR_ERR_INVALID_ARG, "bad vr_partial entry");
        if (((uintptr_t)p.d_data & (mode == VR_MODE_EA ? 15 : 3)) != 0)
            return fail(ctx, VR_ERR_INVALID_ARG, "vr_partial.d_data misaligned");
    }
    constexpr int kStage = 128;                              // descriptors converted per copy, on the stack: no host allocation
    PartialDev stage[kStage];
    for (int first = 0; first < n; first += kStage) {
        const int cnt = std::min(kStage, n - first);
        for (int i = 0; i < cnt; ++i) {
            const vr_partial& p = hp[first + i];
            PartialDev& d = stage[i];
            d.brick = p.brick; d.b[0] = d.b[1] = d.b[2] = 0; d.otile0 = 0;   // the fold reads rectangles and pixels only
            d.x0 = p.x0; d.y0 = p.y0; d.w = p.w; d.h = p.h; d.tile0 = 0;
            d.pitch = (long long)p.pitch_px; d.data = p.d_data;
        }
        VR_CUDA(ctx, static_partials_store(first, stage, cnt, s));
    }
    VR_CUDA(ctx, launch_composite_static(ctx->view, mode, n, d_out, bg, s));
    ctx->launches += 1;
    return VR_OK;
}

int vr_ipc_export(vr_ctx* ctx, const void* d_ptr, unsigned char handle[64], size_t* offset) {
    if (!ctx) return VR_ERR_INVALID_ARG;
    enter(ctx);
    if (!d_ptr || !handle || !offset) return fail(ctx, VR_ERR_INVALID_ARG, "vr_ipc_export: bad argument");
    static_assert(sizeof(cudaIpcMemHandle_t) == 64, "cudaIpcMemHandle_t is 64 bytes");
    cudaIpcMemHandle_t h;
    VR_CUDA(ctx, cudaIpcGetMemHandle(&h, const_cast<void*>(d_ptr)));       // names the whole allocation d_ptr lies in
    // the base of that allocation: a driver call, looked up at run time so that libvr needs no link to libcuda
    typedef CUresult (*range_fn)(CUdeviceptr*, size_t*, CUdeviceptr);
    void* fn = nullptr;
    cudaDriverEntryPointQueryResult qr;
    VR_CUDA(ctx, cudaGetDriverEntryPoint("cuMemGetAddressRange", &fn, cudaEnableDefault, &qr));
    CUdeviceptr base = 0;
    size_t size = 0;
    if (!fn || qr != cudaDriverEntryPointSuccess || ((range_fn)fn)(&base, &size, (CUdeviceptr)d_ptr) != CUDA_SUCCESS)
        return fail(ctx, VR_ERR_CUDA, "vr_ipc_export: cuMemGetAddressRange failed");
    std::memcpy(handle, &h, 64);
    *offset = (size_t)((CUdeviceptr)d_ptr - base);
    return VR_OK;
}

int vr_ipc_open(vr_ctx* ctx, const unsigned char handle[64], size_t offset, void** d_ptr) {
    if (!ctx) return VR_ERR_INVALID_ARG;
    enter(ctx);
    if (!handle || !d_ptr) return fail(ctx, VR_ERR_INVALID_ARG, "vr_ipc_open: bad argument");
    cudaIpcMemHandle_t h;
    std::memcpy(&h, handle, 64);
    void* base = nullptr;
    VR_CUDA(ctx, cudaIpcOpenMemHandle(&base, h, cudaIpcMemLazyEnablePeerAccess));
    ctx->ipc_bases.push_back(base);                                          // closed by vr_destroy
    *d_ptr = (char*)base + offset;
    return VR_OK;
}

int vr_fold_peers(vr_ctx* ctx, int mode, const void* const* h_d_frames, const int* h_order, int n, int width, int height,
                  size_t pitch_px, int y0, int rows, void* const* h_d_out, int n_out, size_t out_pitch_px, const float bg[4],
                  void* stream) {
    VR_RANGE();
    if (!ctx) return VR_ERR_INVALID_ARG;
    enter(ctx);
    if (!h_d_frames || !h_order || !h_d_out || !bg || n <= 0 || n > kMaxPeers || n_out <= 0 || n_out > kMaxPeers || width <= 0 ||
        height <= 0 || pitch_px < (size_t)width || out_pitch_px < (size_t)width || y0 < 0 || rows < 0 || y0 + rows > height ||
        (mode != VR_MODE_MIP && mode != VR_MODE_EA))
        return fail(ctx, VR_ERR_INVALID_ARG, "vr_fold_peers: bad argument");
    PeerList L{};
    const uintptr_t align = mode == VR_MODE_EA ? 15 : 3;
    for (int g = 0; g < n; ++g) {
        const int r = h_order[g];
        if (r < 0 || r >= n || !h_d_frames[r] || ((uintptr_t)h_d_frames[r] & align)) return fail(ctx, VR_ERR_INVALID_ARG, "vr_fold_peers: bad order / frame pointer");
        L.in[g] = h_d_frames[r];
    }
    for (int o = 0; o < n_out; ++o) {
        if (!h_d_out[o] || ((uintptr_t)h_d_out[o] & align)) return fail(ctx, VR_ERR_INVALID_ARG, "vr_fold_peers: bad output pointer");
        L.out[o] = h_d_out[o];
    }
    L.n = n; L.n_out = n_out;
    VR_CUDA(ctx, launch_fold_peers(L, mode, width, (long long)pitch_px, y0, rows, (long long)out_pitch_px, bg, (cudaStream_t)stream));
    ctx->launches += rows > 0 ? 1 : 0;
    return VR_OK;
}

int vr_touch_layout(vr_ctx* ctx, size_t* bitmap_bytes) {
    if (!ctx || !bitmap_bytes) return VR_ERR_INVALID_ARG;
    enter(ctx);
    if (!ctx->has_cube) return fail(ctx, VR_ERR_STATE, "no cube");
    const size_t sectors = cube_bytes(ctx->cube) / 32;
    *bitmap_bytes = align_up((sectors + 7) / 8, 256);
    return VR_OK;
}

int vr_measure_touch(vr_ctx* ctx, int mode, const vr_partial* hp, int n, float tau, void* d_bitmap, int accumulate, void* stream) {
    VR_RANGE();
    int rc = check_render_state(ctx, mode == VR_MODE_EA);
    if (rc) return rc;
    if (n < 0 || (n > 0 && !hp) || (mode != VR_MODE_MIP && mode != VR_MODE_EA) || !(tau > 0.f) || !d_bitmap || ((uintptr_t)d_bitmap & 3) != 0)
        return fail(ctx, VR_ERR_INVALID_ARG, "vr_measure_touch: bad argument");
    cudaStream_t s = (cudaStream_t)stream;
    if ((rc = ensure_tables(ctx, s))) return rc;
    int tiles = 0;
    if ((rc = upload_partials(ctx, mode, hp, n, true, &tiles, s))) return rc;
    RenderArgs a{};
    a.mode = mode; a.tau = mode == VR_MODE_EA ? tau : 2.f; a.skip = skip_level(ctx, a.mode, true); a.variant = pick_variant(ctx, a.mode, a.skip);
    a.dense = resolve_dense(ctx); a.ring = resolve_ring(ctx, a.mode);
    if ((rc = ensure_occ(ctx, a.skip, s))) return rc;
    size_t bytes = 0;
    vr_touch_layout(ctx, &bytes);
    if (!accumulate) {
        VR_CUDA(ctx, cudaMemsetAsync(d_bitmap, 0, bytes, s));
        VR_CUDA(ctx, cudaMemsetAsync(ctx->d_scratch + 2, 0, sizeof(unsigned long long), s));
    }
    VR_CUDA(ctx, launch_touch(ctx->cube, ctx->view, tf_desc(ctx), a, ctx->d_partials, n, tiles, (unsigned*)d_bitmap, ctx->d_scratch + 2, s));
    ctx->launches += (n > 0 && tiles > 0) ? 1 : 0;
    return VR_OK;
}

int vr_touch_count(vr_ctx* ctx, const void* d_bitmap, uint64_t out[3], void* stream) {
    VR_RANGE();
    if (!ctx || !d_bitmap || !out) return VR_ERR_INVALID_ARG;
    enter(ctx);
    if (!ctx->has_cube) return fail(ctx, VR_ERR_STATE, "no cube");
    cudaStream_t s = (cudaStream_t)stream;
    size_t bytes = 0;
    vr_touch_layout(ctx, &bytes);
    VR_CUDA(ctx, cudaMemsetAsync(ctx->d_scratch, 0, 2 * sizeof(unsigned long long), s));
    VR_CUDA(ctx, launch_touch_count((const unsigned*)d_bitmap, (long long)(bytes / 4), ctx->d_scratch, s));
    ctx->launches += 1;
    unsigned long long h[3];
    VR_CUDA(ctx, cudaMemcpyAsync(h, ctx->d_scratch, sizeof(h), cudaMemcpyDeviceToHost, s));
    VR_CUDA(ctx, cudaStreamSynchronize(s));
    out[0] = h[0]; out[1] = h[1]; out[2] = h[2];
    return VR_OK;
}

int vr_get_counters(vr_ctx* ctx, vr_counters* out, void* stream) {
    VR_RANGE();
    if (!ctx || !out) return VR_ERR_INVALID_ARG;
    enter(ctx);
    unsigned long long h[kNumCounters];
    cudaStream_t s = (cudaStream_t)stream;
    VR_CUDA(ctx, cudaMemcpyAsync(h, ctx->d_counters, sizeof(h), cudaMemcpyDeviceToHost, s));
    VR_CUDA(ctx, cudaStreamSynchronize(s));
    out->rays = (int64_t)h[kRays]; out->nominal_samples = (int64_t)h[kNominal]; out->taken_samples = (int64_t)h[kTaken];
    out->bricks_visited = (int64_t)h[kVisited]; out->bricks_skipped = (int64_t)h[kSkipped];
    out->rays_terminated = (int64_t)h[kTerminated]; out->kernel_launches = ctx->launches;
    return VR_OK;
}

int vr_reset_counters(vr_ctx* ctx, void* stream) {
    if (!ctx) return VR_ERR_INVALID_ARG;
    enter(ctx);
    VR_CUDA(ctx, cudaMemsetAsync(ctx->d_counters, 0, kNumCounters * sizeof(unsigned long long), (cudaStream_t)stream));
    ctx->launches = 0;
    return VR_OK;
}

int vr_overlay_catalogue(vr_ctx* ctx, const vr_catalogue* cat, float* d_frame_rgba, int* d_pick, void* stream) {
    VR_RANGE();
    if (!ctx) return VR_ERR_INVALID_ARG;
    enter(ctx);
    if (!ctx->has_view) return fail(ctx, VR_ERR_STATE, "no view: call vr_set_view first");
    if (!cat || !d_pick || cat->n < 0 || (cat->n > 0 && (!cat->d_boxes || (d_frame_rgba && !cat->d_colours))))
        return fail(ctx, VR_ERR_INVALID_ARG, "vr_overlay_catalogue: bad argument");
    if (d_frame_rgba && ((uintptr_t)d_frame_rgba & 15) != 0) return fail(ctx, VR_ERR_INVALID_ARG, "vr_overlay_catalogue: frame must be 16-byte aligned");
    VR_CUDA(ctx, launch_overlay(ctx->view, ctx->M, cat->d_boxes, cat->d_colours, cat->d_visible, cat->n, d_frame_rgba, d_pick,
                                (cudaStream_t)stream));
    ctx->launches += cat->n > 0 ? (d_frame_rgba ? 3 : 2) : 1;
    return VR_OK;
}

int vr_overlay_pick(vr_ctx* ctx, const int* d_pick, int x, int y, int radius, int* box, void* stream) {
    VR_RANGE();
    if (!ctx) return VR_ERR_INVALID_ARG;
    enter(ctx);
    if (!ctx->has_view) return fail(ctx, VR_ERR_STATE, "no view: call vr_set_view first");
    if (!d_pick || !box || radius < 0 || radius > 64) return fail(ctx, VR_ERR_INVALID_ARG, "vr_overlay_pick: bad argument");
    cudaStream_t s = (cudaStream_t)stream;
    int* d_out = reinterpret_cast<int*>(ctx->d_scratch);
    VR_CUDA(ctx, launch_overlay_pick(ctx->view, d_pick, x, y, radius, d_out, s));
    ctx->launches += 1;
    VR_CUDA(ctx, cudaMemcpyAsync(box, d_out, sizeof(int), cudaMemcpyDeviceToHost, s));
    VR_CUDA(ctx, cudaStreamSynchronize(s));
    return VR_OK;
}

int vr_pyramid_layout(int width, int height, int tile, int* n_levels, vr_pyramid_level* levels, size_t* bytes) {
    if (width <= 0 || height <= 0 || tile < 16 || tile > 4096 || (tile & (tile - 1)) != 0 || !n_levels || !levels || !bytes) return VR_ERR_INVALID_ARG;
    const int n = pyramid_levels(width, height, tile, levels, bytes);
    if (n < 0) return VR_ERR_INVALID_ARG;
    *n_levels = n;
    return VR_OK;
}

int vr_build_pyramid(vr_ctx* ctx, const float* d_frame_rgba, int width, int height, size_t pitch_px, int tile, void* d_out, void* stream) {
    VR_RANGE();
    if (!ctx) return VR_ERR_INVALID_ARG;
    enter(ctx);
    if (!d_frame_rgba || !d_out || width <= 0 || height <= 0 || pitch_px < (size_t)width || tile < 16 || tile > 4096 ||
        (tile & (tile - 1)) != 0 || ((uintptr_t)d_frame_rgba & 15) != 0 || ((uintptr_t)d_out & 3) != 0)
        return fail(ctx, VR_ERR_INVALID_ARG, "vr_build_pyramid: bad argument");
    int launches = 0;
    cudaError_t e = launch_pyramid(d_frame_rgba, width, height, (long long)pitch_px, tile, d_out, &launches, (cudaStream_t)stream);
    ctx->launches += launches;
    if (e != cudaSuccess) return cuda_fail(ctx, e, "vr_build_pyramid");
    return VR_OK;
}

int vr_get_plan(vr_ctx* ctx, int mode, int out[3], void* stream) {
    VR_RANGE();
    int rc = check_render_state(ctx, mode == VR_MODE_EA);
    if (rc) return rc;
    if (!out || (mode != VR_MODE_MIP && mode != VR_MODE_EA)) return fail(ctx, VR_ERR_INVALID_ARG, "vr_get_plan: bad argument");
    if ((rc = ensure_tables(ctx, (cudaStream_t)stream))) return rc;
    out[1] = skip_level(ctx, mode, true); out[0] = use_mip_tiles(ctx, mode) ? 5 : pick_variant(ctx, mode, out[1]); out[2] = mode == VR_MODE_EA ? resolve_dense(ctx) : 0;
    return VR_OK;
}

int vr_set_option(vr_ctx* ctx, int option, int value) {
    if (!ctx) return VR_ERR_INVALID_ARG;
    if (option == VR_OPT_SKIP) { ctx->opt_skip = value ? 1 : 0; return VR_OK; }
    if (option == VR_OPT_CELL_SKIP) { ctx->opt_cell_skip = value < 0 ? -1 : (value ? 1 : 0); return VR_OK; }
    if (option == VR_OPT_LAYOUT) {
        if (value != 0 && value != 1) return fail(ctx, VR_ERR_INVALID_ARG, "vr_set_option: layout must be 0 (rows) or 1 (4x4x2 blocks)");
        if (value == 0 && ctx->opt_vtype == 1) return fail(ctx, VR_ERR_INVALID_ARG, "vr_set_option: float16 voxels need the micro-block layout");
        ctx->opt_layout = value; return VR_OK;                  // takes effect at the next upload / generate / attach
    }
    if (option == VR_OPT_L2_FETCH) {
        if (value != 32 && value != 64 && value != 128) return fail(ctx, VR_ERR_INVALID_ARG, "vr_set_option: L2 fetch granularity must be 32, 64 or 128");
        VR_CUDA(ctx, cudaDeviceSetLimit(cudaLimitMaxL2FetchGranularity, (size_t)value));
        return VR_OK;
    }
    if (option == VR_OPT_VOXEL_TYPE) {
        if (value != 0 && value != 1) return fail(ctx, VR_ERR_INVALID_ARG, "vr_set_option: voxel type must be 0 (float32) or 1 (float16)");
        if (value == 1 && ctx->opt_layout != 1) return fail(ctx, VR_ERR_INVALID_ARG, "vr_set_option: float16 voxels need the micro-block layout (VR_OPT_LAYOUT 1)");
        ctx->opt_vtype = value; return VR_OK;                   // takes effect at the next upload / generate / attach
    }
    if (option == VR_OPT_RING) { ctx->opt_ring = value < 0 ? -1 : (value ? 1 : 0); return VR_OK; }
    if (option == VR_OPT_MIP_TILES) { ctx->opt_mip_tiles = value < 0 ? -1 : (value ? 1 : 0); return VR_OK; }
    if (option == VR_OPT_OCCUPANCY) { ctx->opt_occ = value < 0 ? -1 : (value ? 1 : 0); return VR_OK; }
    if (option == VR_OPT_DENSE) { ctx->opt_dense = value < 0 ? -1 : (value ? 1 : 0); return VR_OK; }
    if (option == VR_OPT_VARIANT) {
        if (value != -1 && value != 0 && value != 1 && value != 3 && value != 4) return fail(ctx, VR_ERR_INVALID_ARG, "vr_set_option: unknown marcher variant");
        ctx->opt_variant = value; return VR_OK;
    }
    return fail(ctx, VR_ERR_INVALID_ARG, "vr_set_option: unknown option");
}

}  // extern "C"
