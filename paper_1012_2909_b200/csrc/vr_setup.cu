// Set-up passes over the resident cube (SURVEY.md 8(a) S0 metadata and S1 classification; O-10), written as
// line-granular streaming kernels: the brick-major cube is a sequence of 128-byte lines (one 4 x 4 x 2
// micro-block each, layout 1), so every pass reads whole lines, coalesced, once.
//
//  cell_minmax_lines_kernel  (min,max) per 8^3 macro-cell incl. its +1 halo layer: one CTA per row of cells
//                            along x, its warps stream the 15 columns of micro-blocks the row needs.
//  hot_kernel                per transfer function: one bit per voxel, "this voxel maps above the table's
//                            transparent prefix"; the cube streams through shared memory in bulk asynchronous
//                            copies (cp.async.bulk + mbarrier ring), one ballot per line.
//  dilate_kernel             occupancy bit of a trilinear cell = OR of the hot bits of its 8 corners: pure bit
//                            operations on the hot words of the 8 neighbouring micro-blocks.
//  classify_cells_kernel     the same O-10 test per macro-cell from its (min,max).
#include "vr_async.cuh"
#include "vr_sample.cuh"

namespace vr {

namespace {

// ---------------------------------------------------------------------------------------------- S0: cell (min,max)
constexpr int kMMWarps = 8;
constexpr int kMMCells = 64;       // cells of one row handled per CTA (256^3 bricks: 32)

// Column j of the 3 x 5 columns of micro-blocks (rows of lines along x) that a row of cells (cy, cz) needs:
// ty = 2 cy + j % 3, tz = 4 cz + j / 3; the third column in y and the fifth in z are the +1 halo planes.
// a row of 4 x-voxels of a line as float32
__device__ __forceinline__ float4 load_row(const float* rows, long long i) { return __ldg(reinterpret_cast<const float4*>(rows) + i); }
__device__ __forceinline__ float4 load_row(const __half* rows, long long i) {
    const uint2 u = __ldg(reinterpret_cast<const uint2*>(rows) + i);
    const float2 a = __half22float2(*reinterpret_cast<const __half2*>(&u.x)), b = __half22float2(*reinterpret_cast<const __half2*>(&u.y));
    return make_float4(a.x, a.y, b.x, b.y);
}

template <typename V>
__global__ void __launch_bounds__(kMMWarps * 32)
cell_minmax_lines_kernel(const __grid_constant__ CubeDesc c, int chunks_x) {
    __shared__ float smin[kMMWarps][kMMCells + 1], smax[kMMWarps][kMMCells + 1];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    long long u = blockIdx.x;
    const int xc = (int)(u % chunks_x); u /= chunks_x;
    const int cy = (int)(u % c.C[1]); u /= c.C[1];
    const int cz = (int)(u % c.C[2]); u /= c.C[2];
    const int brick = c.win_lo + (int)u;
    const int bi[3] = {brick % c.G[0], (brick / c.G[0]) % c.G[1], brick / (c.G[0] * c.G[1])};
    int lim[3];                                              // last stored index per axis that is a voxel of the cube (halo included)
#pragma unroll
    for (int a = 0; a < 3; ++a) lim[a] = min(c.B[a], c.N[a] - 1 - bi[a] * c.B[a]);
    const int cx0 = xc * kMMCells, ncell = min(kMMCells, c.C[0] - cx0);
    for (int i = lane; i <= kMMCells; i += 32) { smin[warp][i] = INFINITY; smax[warp][i] = -INFINITY; }
    __syncwarp();
    const V* brick_base = reinterpret_cast<const V*>(c.cube) + (long long)brick * c.stride;
    const int tx_a = 2 * cx0, tx_b = min(c.T[0] - 1, 2 * (cx0 + ncell));     // last line: the halo plane lx = 8 (cx0 + ncell)
    const int r = lane & 7, g = lane >> 3;
    const int ly3 = 2 * (r >> 2) + (r & 1), lz1 = (r >> 1) & 1;                // this lane's row of 4 x-voxels inside a line
    for (int j = warp; j < 15; j += kMMWarps) {
        const int ty_off = j % 3, tz_off = j / 3;
        const int ty = 2 * cy + ty_off, tz = 4 * cz + tz_off;
        if (ty >= c.T[1] || tz >= c.T[2]) continue;
        const int ly = 4 * ty + ly3, lz = 2 * tz + lz1;
        const bool row_ok = ly <= lim[1] && lz <= lim[2] && (ty_off < 2 || ly3 == 0) && (tz_off < 4 || lz1 == 0);
        const V* col = brick_base + 32LL * c.T[0] * (ty + (long long)c.T[1] * tz) + 4 * r;   // rows of 4 voxels, 8 per line
        // group g of 8 lanes takes cell c0 + g: its two lines and the first plane of the next line are reduced inside
        // the lane, so only one reduction over the 8 rows (6 shuffles) is paid per cell; 8 cells (2 KiB) in flight per warp
        auto fold4 = [&](const float4 v, const int x0, float& mn, float& mx) {
            if (x0 + 3 <= lim[0]) {
                mn = fminf(mn, fminf(fminf(v.x, v.y), fminf(v.z, v.w))); mx = fmaxf(mx, fmaxf(fmaxf(v.x, v.y), fmaxf(v.z, v.w)));
            } else {
                if (x0 <= lim[0]) { mn = fminf(mn, v.x); mx = fmaxf(mx, v.x); }
                if (x0 + 1 <= lim[0]) { mn = fminf(mn, v.y); mx = fmaxf(mx, v.y); }
                if (x0 + 2 <= lim[0]) { mn = fminf(mn, v.z); mx = fmaxf(mx, v.z); }
            }
        };
        for (int c0 = 0; c0 < ncell; c0 += 8) {
            float4 va[2], vb[2];
            float vh[2];
#pragma unroll
            for (int u = 0; u < 2; ++u) {
                const int tx = tx_a + 2 * (c0 + 4 * u + g);
                const bool ok = row_ok && c0 + 4 * u + g < ncell;
                va[u] = (ok && tx <= tx_b) ? load_row(col, 8LL * tx) : make_float4(0.f, 0.f, 0.f, 0.f);
                vb[u] = (ok && tx + 1 <= tx_b) ? load_row(col, 8LL * (tx + 1)) : make_float4(0.f, 0.f, 0.f, 0.f);
                vh[u] = (ok && tx + 2 <= tx_b) ? load_voxel(col + 32LL * (tx + 2)) : 0.f;
            }
#pragma unroll
            for (int u = 0; u < 2; ++u) {
                const int cell = c0 + 4 * u + g, tx = tx_a + 2 * cell;
                float mn = INFINITY, mx = -INFINITY;
                if (row_ok && cell < ncell) {
                    if (tx <= tx_b) fold4(va[u], 4 * tx, mn, mx);
                    if (tx + 1 <= tx_b) fold4(vb[u], 4 * tx + 4, mn, mx);
                    if (tx + 2 <= tx_b && 4 * tx + 8 <= lim[0]) { mn = fminf(mn, vh[u]); mx = fmaxf(mx, vh[u]); }
                }
#pragma unroll
                for (int o = 1; o < 8; o <<= 1) {                  // over the 8 rows of the lines
                    mn = fminf(mn, __shfl_xor_sync(0xffffffffu, mn, o)); mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, o));
                }
                if (r == 0 && cell < ncell) {                      // one lane per cell: no two lanes meet in a slot
                    smin[warp][cell] = fminf(smin[warp][cell], mn); smax[warp][cell] = fmaxf(smax[warp][cell], mx);
                }
            }
        }
        __syncwarp();
    }
    __syncthreads();
    for (int i = threadIdx.x; i < ncell; i += kMMWarps * 32) {
        float mn = INFINITY, mx = -INFINITY;
#pragma unroll
        for (int w = 0; w < kMMWarps; ++w) { mn = fminf(mn, smin[w][i]); mx = fmaxf(mx, smax[w][i]); }
        c.cell_mm[(long long)brick * c.cells_per_brick + (cx0 + i) + c.C[0] * (cy + c.C[1] * cz)] = make_float2(mn, mx);
    }
}

// ---------------------------------------------------------------------------------------------- S1: hot bits
constexpr int kHotLines = 64;      // lines per stage (8 KiB)
constexpr int kHotStages = 4;
constexpr int kHotThreads = 256;

// hot[line] bit s = voxel in slot s of the line maps above the transparent prefix: (v - vmin) * scale > thr.
// Persistent CTAs; chunk k of a CTA is chunk blockIdx.x + k * gridDim.x of the window's lines.
template <typename V>
__global__ void __launch_bounds__(kHotThreads)
hot_kernel(const V* __restrict__ lines, unsigned* __restrict__ hot, long long n_lines, float vmin, float scale, float thr) {
    __shared__ __align__(128) V buf[kHotStages][kHotLines * 32];
    __shared__ __align__(8) unsigned long long full[kHotStages];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const long long n_chunks = (n_lines + kHotLines - 1) / kHotLines;
    const long long mine = blockIdx.x < n_chunks ? (n_chunks - 1 - blockIdx.x) / gridDim.x + 1 : 0;
    auto issue = [&](long long k) {                            // thread 0 only
        if (k >= mine) return;
        const long long chunk = blockIdx.x + k * gridDim.x;
        const int s = (int)(k % kHotStages);
        const unsigned nl = (unsigned)min((long long)kHotLines, n_lines - chunk * kHotLines);
        const unsigned bar = (unsigned)__cvta_generic_to_shared(&full[s]);
        mbar_expect_tx(bar, nl * 32u * (unsigned)sizeof(V));
        bulk_load((unsigned)__cvta_generic_to_shared(&buf[s][0]), lines + chunk * kHotLines * 32, nl * 32u * (unsigned)sizeof(V), bar);
    };
    if (threadIdx.x == 0) {
        for (int s = 0; s < kHotStages; ++s) mbar_init((unsigned)__cvta_generic_to_shared(&full[s]), 1u);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    if (threadIdx.x == 0) for (int k = 0; k < kHotStages; ++k) issue(k);
    constexpr int kPerWarp = kHotLines / (kHotThreads / 32);   // 8 consecutive lines per warp
    for (long long k = 0; k < mine; ++k) {
        const int s = (int)(k % kHotStages);
        mbar_wait((unsigned)__cvta_generic_to_shared(&full[s]), (unsigned)((k / kHotStages) & 1));
        const long long chunk = blockIdx.x + k * gridDim.x;
        const int nl = (int)min((long long)kHotLines, n_lines - chunk * kHotLines);
        unsigned word = 0u;
#pragma unroll
        for (int j = 0; j < kPerWarp; ++j) {
            const int line = warp * kPerWarp + j;
            const float v = line < nl ? (float)buf[s][line * 32 + lane] : 0.f;
            const unsigned b = __ballot_sync(0xffffffffu, line < nl && __fmul_rn(__fsub_rn(v, vmin), scale) > thr);
            if (lane == j) word = b;
        }
        if (lane < kPerWarp && warp * kPerWarp + lane < nl) hot[chunk * kHotLines + warp * kPerWarp + lane] = word;
        __syncthreads();                                       // every warp is done with stage s
        if (threadIdx.x == 0) issue(k + kHotStages);
    }
}

// occ word of micro-block (tx, ty, tz), bit = slot of the cell's lower corner inside the block
// (slot = (lx&3) + 4 (ly&1) + 8 (lz&1) + 16 ((ly>>1)&1)): OR of the hot bits of the cell's 8 corners.
__global__ void dilate_kernel(const __grid_constant__ CubeDesc c, const unsigned* __restrict__ hot, long long n_words) {
    const long long per = c.occ_words_per_brick;               // = T0 T1 T2, the lines of a brick
    for (long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x; e < n_words; e += (long long)gridDim.x * blockDim.x) {
        const long long bw = e / per;                          // brick of the window
        const int mb = (int)(e % per);
        const int tx = mb % c.T[0], ty = (mb / c.T[0]) % c.T[1], tz = mb / (c.T[0] * c.T[1]);
        const unsigned* H = hot + bw * per;
        const bool hx = tx + 1 < c.T[0], hy = ty + 1 < c.T[1], hz = tz + 1 < c.T[2];
        auto at = [&](int dx, int dy, int dz) -> unsigned {
            if ((dx && !hx) || (dy && !hy) || (dz && !hz)) return 0u;     // no such block: its voxels lie beyond the halo
            return __ldg(H + mb + dx + c.T[0] * (dy + c.T[1] * dz));
        };
        auto along_x = [&](int dy, int dz) -> unsigned {
            const unsigned h = at(0, dy, dz);
            return h | ((h >> 1) & 0x77777777u) | ((at(1, dy, dz) << 3) & 0x88888888u);
        };
        auto along_xy = [&](int dz) -> unsigned {
            const unsigned a = along_x(0, dz), a1 = along_x(1, dz);
            // ly&3: 0 -> 1 and 2 -> 3 are 4 slots up, 1 -> 2 is 12 up, 3 -> 0 of the next block is 20 down
            return a | ((a >> 4) & 0x0F0F0F0Fu) | ((a >> 12) & 0x0000F0F0u) | ((a1 << 20) & 0xF0F00000u);
        };
        const unsigned b0 = along_xy(0), b1 = along_xy(1);
        (c.occ + (long long)c.win_lo * per)[e] = b0 | ((b0 >> 8) & 0x00FF00FFu) | ((b1 << 8) & 0xFF00FF00u);
    }
}

// ---------------------------------------------------------------------------------------------- S1: macro-cells
// O-10 per transfer function: one bit per 8^3 macro-cell, set iff a table entry that the cell's
// value range [min, max] (halo-inclusive) can touch has non-zero opacity.  `nz` is the running
// count of entries with non-zero baked opacity, so the range test is one subtraction.
struct NzPrefix { int v[257]; };
__global__ void classify_cells_kernel(const __grid_constant__ CubeDesc c, const __grid_constant__ NzPrefix nz,
                                      float vmin, float scale, long long n_slots,
                                      unsigned long long* __restrict__ active_count) {
    for (long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x; e < n_slots;
         e += (long long)gridDim.x * blockDim.x) {
        const long long word = (long long)c.win_lo * c.cell_words_per_brick + (e >> 5);
        const int brick = (int)(word / c.cell_words_per_brick);
        const int cidx = (int)(word % c.cell_words_per_brick) * 32 + (int)(e & 31);
        bool active = false;
        if (cidx < c.cells_per_brick) {
            const float2 mm = c.cell_mm[(long long)brick * c.cells_per_brick + cidx];
            if (mm.x <= mm.y) {
                float xa = fminf(fmaxf(__fmul_rn(__fsub_rn(mm.x, vmin), scale), 0.f), 255.f);
                float xb = fminf(fmaxf(__fmul_rn(__fsub_rn(mm.y, vmin), scale), 0.f), 255.f);
                const int lo = max(0, min((int)floorf(xa), 255)), hi = max(0, min((int)ceilf(xb), 255));
                active = nz.v[hi + 1] - nz.v[lo] > 0;
            }
        }
        const unsigned bits = __ballot_sync(0xffffffffu, active);
        if ((e & 31) == 0) {
            c.cell_bits[word] = bits;
            if (bits) atomicAdd(active_count, (unsigned long long)__popc(bits));
        }
    }
}

struct HalfTable { float4 v[128]; };
__global__ void upload_half_kernel(float4* dst, const __grid_constant__ HalfTable h, int offset) {
    if (threadIdx.x < 128) dst[offset + threadIdx.x] = h.v[threadIdx.x];
}

}  // namespace

cudaError_t launch_cell_minmax_lines(const CubeDesc& c, cudaStream_t s) {
    const int chunks_x = (c.C[0] + kMMCells - 1) / kMMCells;
    const long long ctas = (long long)(c.win_hi - c.win_lo) * c.C[2] * c.C[1] * chunks_x;
    if (ctas <= 0) return cudaSuccess;
    if (ctas > 0x7fffffffLL) return cudaErrorInvalidConfiguration;
    if (c.vtype == 1) cell_minmax_lines_kernel<__half><<<(unsigned)ctas, kMMWarps * 32, 0, s>>>(c, chunks_x);
    else cell_minmax_lines_kernel<float><<<(unsigned)ctas, kMMWarps * 32, 0, s>>>(c, chunks_x);
    return cudaGetLastError();
}

// Occupancy bits against a table whose entries 0 .. t are transparent (thr = t): hot pass over the cube, then dilation.
cudaError_t launch_classify_occ(const CubeDesc& c, float vmin, float scale, float thr, cudaStream_t s) {
    const long long n_lines = (long long)(c.win_hi - c.win_lo) * c.occ_words_per_brick;
    if (n_lines <= 0) return cudaSuccess;
    unsigned* hot = c.hot + (long long)c.win_lo * c.occ_words_per_brick;
    if (c.vtype == 1) hot_kernel<__half><<<148 * 4, kHotThreads, 0, s>>>(reinterpret_cast<const __half*>(c.cube) + (long long)c.win_lo * c.stride, hot, n_lines, vmin, scale, thr);
    else hot_kernel<float><<<148 * 4, kHotThreads, 0, s>>>(c.cube + (long long)c.win_lo * c.stride, hot, n_lines, vmin, scale, thr);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    dilate_kernel<<<148 * 16, 256, 0, s>>>(c, hot, n_lines);
    return cudaGetLastError();
}

cudaError_t launch_classify_cells(const CubeDesc& c, const int nz_prefix[257], float vmin, float scale,
                                  unsigned long long* d_active_count, cudaStream_t s) {
    NzPrefix nz;
    for (int i = 0; i < 257; ++i) nz.v[i] = nz_prefix[i];
    const long long n_slots = (long long)(c.win_hi - c.win_lo) * c.cell_words_per_brick * 32;
    long long blocks = (n_slots + 255) / 256;
    if (blocks > 148LL * 32) blocks = 148LL * 32;
    if (blocks <= 0) return cudaSuccess;
    classify_cells_kernel<<<(int)blocks, 256, 0, s>>>(c, nz, vmin, scale, n_slots, d_active_count);
    return cudaGetLastError();
}

// The 4 KiB table travels in kernel parameter space (copied at launch), so the host buffer can be
// reused immediately and no pinned staging or stream synchronisation is needed.
cudaError_t launch_upload_table(float4* d_dst, const float* h_src_1024, cudaStream_t s) {
    for (int half = 0; half < 2; ++half) {
        HalfTable h;
        for (int i = 0; i < 128; ++i) {
            const float* p = h_src_1024 + 4 * (128 * half + i);
            h.v[i] = make_float4(p[0], p[1], p[2], p[3]);
        }
        upload_half_kernel<<<1, 128, 0, s>>>(d_dst, h, 128 * half);
        cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) return e;
    }
    return cudaSuccess;
}

}  // namespace vr
