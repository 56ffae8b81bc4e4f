// The ray marcher (BASELINE.json north_star (2)): per-pixel rays through the
// brick-major cube, fixed step, trilinear interpolation, MIP or front-to-back emission-absorption
// through the 256-entry transfer function with early ray termination, min/max brick skipping.
//
// Arithmetic contract (readings O-2...O-7, O-11): the
// ray is set up in fp64 and rounded once to float32; every per-sample operation is an explicit
// IEEE float32 + - * fma floor min max compare (no fast-math, built with --fmad=false), so frames
// agree with the float32 instantiation of the oracle to the bit and with its fp64 instantiation
// within BASELINE.json's tolerances.
#pragma once
#include <type_traits>

#include "vr_sample.cuh"

namespace vr {

namespace {

// ================================================================== variant 0: one ray per thread
// March the lattice samples k .. ke (all of them members of brick `bid`, O-3) into `acc`.  With
// A.skip >= 2 the interval is cut into runs inside 8^3 macro-cells and idle runs are jumped.
// Returns true if early ray termination fired.
template <int MODE, int LAYOUT, bool JUMP = false, typename VT = float>
__device__ __forceinline__ bool march_interval(const CubeDesc& c, const Ray& r, const TFDesc& T, const RenderArgs& A,
                                               const float4* tab, int bid, const int lo[3], int k, int ke,
                                               Accum& acc, Stats& st) {
    BrickRefT<VT> b = brick_ref<LAYOUT, VT>(c, bid, lo);
    const unsigned* occ = (MODE == VR_MODE_EA && LAYOUT == 1 && A.skip >= 3) ? c.occ + (long long)bid * c.occ_words_per_brick : nullptr;
    asm volatile("" : "+l"(b.base), "+l"(occ));             // both stay in registers (else re-derived from the brick id per sample)
    const int S8[3] = {kCell, kCell, kCell};
    // a jump out of an idle micro-block costs about as much as testing 3 samples one by one: worth it when
    // the block holds more than that (measured: step 0.25 -> C4 29.6 to 26.2 ms; step 0.5 -> C2 0.70 to 0.76 ms),
    // and a separate instantiation, because the extra path costs the other one registers
    const bool block_jumps = JUMP && occ != nullptr;        // JUMP kernels are launched for steps < kJumpStep only
    float kf = (float)k;                                    // exact: k < 2^24
    while (k <= ke) {
        int n = ke - k + 1;
        if (A.skip >= 2) {
            // A loop of its own over the idle runs: the lanes of a warp meet again behind it, each at the start
            // of an ACTIVE run (or at the end of its interval), and take the samples below together.  In one
            // loop with the samples, a lane in an idle run would wait for the lanes sampling, then sample alone.
            for (;;) {
                float p[3], fl;
                position(r, kf, p);
                const int iv[3] = {floor_pos(p[0], fl), floor_pos(p[1], fl), floor_pos(p[2], fl)};
                const int clo[3] = {lo[0] + (((iv[0] - lo[0]) >> 3) << 3), lo[1] + (((iv[1] - lo[1]) >> 3) << 3),
                                    lo[2] + (((iv[2] - lo[2]) >> 3) << 3)};
                n = min(ke - k + 1, run_length(r, p, clo, S8));
                if (!cell_idle<MODE>(c, bid, lo, iv[0], iv[1], iv[2], acc.m)) break;
                k += n; kf = __fadd_rn(kf, (float)n); ++st.skip;
                if (k > ke) { n = 0; break; }
            }
            if (n == 0) break;
        }
        ++st.visit;
        if (JUMP && block_jumps) {
            // small steps: inside an active macro-cell the ray leaves every idle 4 x 4 x 2 block of cells (occupancy
            // word == 0) in one jump instead of testing its samples one by one
            for (const int e = k + n; k < e;) {
                float p[3], fl;
                position(r, kf, p);
                const unsigned lx = (unsigned)(floor_pos(p[0], fl) - lo[0]), ly = (unsigned)(floor_pos(p[1], fl) - lo[1]),
                               lz = (unsigned)(floor_pos(p[2], fl) - lo[2]);
                const unsigned word = __ldg(occ + occ_word_index(c, lx, ly, lz));
                if (word == 0u) {
                    const int blo[3] = {lo[0] + (int)(lx & ~3u), lo[1] + (int)(ly & ~3u), lo[2] + (int)(lz & ~1u)};
                    const int S4[3] = {4, 4, 2};
                    const int m = min(run_length(r, p, blo, S4), e - k);
                    k += m; kf = __fadd_rn(kf, (float)m);
                    continue;
                }
                if ((word >> occ_bit_index(lx, ly, lz)) & 1u) {
                    const float v = sample<LAYOUT>(b, p);
                    ++st.taken;
                    if (fold<MODE>(acc, v, tab, T, A.tau)) return true;
                }
                ++k; kf = __fadd_rn(kf, 1.f);
            }
            continue;
        }
        for (const int e = k + n; k < e; ++k, kf = __fadd_rn(kf, 1.f)) {
            float p[3];
            position(r, kf, p);
            if (occ) {                                      // O-10 per trilinear cell: the sample's occupancy bit
                float fl;
                const unsigned lx = (unsigned)(floor_pos(p[0], fl) - lo[0]), ly = (unsigned)(floor_pos(p[1], fl) - lo[1]),
                               lz = (unsigned)(floor_pos(p[2], fl) - lo[2]);
                if (((__ldg(occ + occ_word_index(c, lx, ly, lz)) >> occ_bit_index(lx, ly, lz)) & 1u) == 0u) continue;
            }
            const float v = sample<LAYOUT>(b, p);
            ++st.taken;
            if (fold<MODE>(acc, v, tab, T, A.tau)) return true;
        }
    }
    return false;
}

__device__ __forceinline__ float4 raw_tf_at(const TFDesc& T, float m) {
    float x = __fmul_rn(__fsub_rn(m, T.vmin), T.scale);
    return tf_at(T.raw, x);
}

template <int MODE>
__device__ __forceinline__ void write_frame_pixel(const ViewDesc& V, const TFDesc& T, const RenderArgs& A, int i, int j,
                                                  const Accum& acc, bool any) {
    const long long px = (long long)(V.vy0 + j) * V.pitch + (V.vx0 + i);
    if (MODE == VR_MODE_MIP) {
        A.out[px] = any ? acc.m : A.miss;
        if (A.out_rgba)
            reinterpret_cast<float4*>(A.out_rgba)[px] = any ? raw_tf_at(T, acc.m) : make_float4(0.f, 0.f, 0.f, 0.f);
    } else {                                               // O-7: premultiplied colour over bg
        const float t = __fsub_rn(1.f, acc.A);
        reinterpret_cast<float4*>(A.out)[px] = make_float4(__fmaf_rn(t, A.bg[0], acc.C[0]), __fmaf_rn(t, A.bg[1], acc.C[1]),
                                                           __fmaf_rn(t, A.bg[2], acc.C[2]), __fmaf_rn(t, A.bg[3], acc.A));
    }
}

// ---------------------------------------------------------------- whole frame, O-8 GLOBAL
template <int MODE, int LAYOUT, bool JUMP = false, typename VT = float>
__global__ void __launch_bounds__(kThreads)
render_global_kernel(const __grid_constant__ CubeDesc c, const __grid_constant__ ViewDesc V,
                     const __grid_constant__ TFDesc T, const __grid_constant__ RenderArgs A) {
    __shared__ float4 tab[256];
    if (MODE == VR_MODE_EA) load_tf(tab, T.baked);
    int tx, ty; tile_pixel(tx, ty);
    const int i = blockIdx.x * kTileW + tx, j = blockIdx.y * kTileH + ty;
    const bool live = i < V.W && j < V.H;
    Ray r; r.k0 = 0; r.k1 = -1;
    if (live) setup_ray(V, c, i, j, r);
    Accum acc = {{0.f, 0.f, 0.f}, 0.f, -INFINITY};
    Stats st = {0, 0, 0};
    bool stopped = false;
    int k = r.k0;
    while (k <= r.k1) {
        float p[3];
        position(r, (float)k, p);
        float fl;
        int iv[3] = {floor_pos(p[0], fl), floor_pos(p[1], fl), floor_pos(p[2], fl)};
        int b[3]; brick_of(c, iv, b);
        int lo[3] = {b[0] * c.B[0], b[1] * c.B[1], b[2] * c.B[2]};
        int n = min(run_length(r, p, lo, c.B), r.k1 - k + 1);
        const int bid = b[0] + c.G[0] * (b[1] + c.G[1] * b[2]);
        bool skip = false;
        if (A.skip) {
            if (MODE == VR_MODE_MIP) skip = c.brick_mm[bid].y <= acc.m;       // O-10 (exact)
            else skip = c.brick_active[bid] == 0;
        }
        if (skip) { k += n; ++st.skip; continue; }
        if (march_interval<MODE, LAYOUT, JUMP, VT>(c, r, T, A, tab, bid, lo, k, k + n - 1, acc, st)) { stopped = true; break; }
        k += n;
    }
    if (live) write_frame_pixel<MODE>(V, T, A, i, j, acc, r.k1 >= r.k0);
    if (A.counters) {
        const unsigned long long nom = r.k1 >= r.k0 ? (unsigned long long)(r.k1 - r.k0 + 1) : 0ULL;
        count(A.counters, kRays, nom ? 1 : 0);
        count(A.counters, kNominal, nom);
        count(A.counters, kTaken, st.taken);
        count(A.counters, kVisited, st.visit);
        count(A.counters, kSkipped, st.skip);
        count(A.counters, kTerminated, stopped ? 1 : 0);
    }
}

// ---------------------------------------------------------------- per-brick partial images (O-8 SORT-LAST)
template <int MODE, int LAYOUT, typename VT = float>
__global__ void __launch_bounds__(kThreads)
render_bricks_kernel(const __grid_constant__ CubeDesc c, const __grid_constant__ ViewDesc V,
                     const __grid_constant__ TFDesc T, const __grid_constant__ RenderArgs A,
                     const PartialDev* __restrict__ parts, int n_parts) {
    __shared__ float4 tab[256];
    __shared__ PartialDev part;
    int lx, ly;
    const bool live = locate_tile(parts, n_parts, part, lx, ly);
    if (MODE == VR_MODE_EA) load_tf(tab, T.baked);
    Ray r; r.k0 = 0; r.k1 = -1;
    if (live) setup_ray(V, c, part.x0 + lx, part.y0 + ly, r);
    const int bid = part.brick;
    const int b[3] = {part.b[0], part.b[1], part.b[2]};
    const int lo[3] = {b[0] * c.B[0], b[1] * c.B[1], b[2] * c.B[2]};
    int ka = r.k0, kb = r.k1;
    brick_interval(c, r, b, lo, ka, kb);
    Accum acc = {{0.f, 0.f, 0.f}, 0.f, -INFINITY};
    Stats st = {0, 0, 0};
    const bool stopped = march_interval<MODE, LAYOUT, false, VT>(c, r, T, A, tab, bid, lo, ka, kb, acc, st);
    if (live) {
        const long long px = (long long)ly * part.pitch + lx;
        if (MODE == VR_MODE_MIP) reinterpret_cast<float*>(part.data)[px] = acc.m;
        else reinterpret_cast<float4*>(part.data)[px] = make_float4(acc.C[0], acc.C[1], acc.C[2], acc.A);
    }
    if (A.counters) {
        count(A.counters, kNominal, kb >= ka ? (unsigned long long)(kb - ka + 1) : 0ULL);
        count(A.counters, kTaken, st.taken);
        count(A.counters, kVisited, st.visit);
        count(A.counters, kSkipped, st.skip);
        count(A.counters, kTerminated, stopped ? 1 : 0);
    }
}

// The same partial images, one CTA per PIXEL TILE of the view instead of one per (brick, tile): the
// ray of a pixel is set up once (fp64) and reused for every brick whose screen rectangle holds
// the pixel (dense rays cross 10-30 bricks: on C4 the per-brick set-up was a fifth of all
// instructions).  The CTA culls the partial rectangles against its tile into a shared bitmask
// (as composite_kernel does) and takes the hits one after the other.
constexpr int kCullChunk = 2048;

template <int MODE, int LAYOUT, bool JUMP, typename VT = float>
__global__ void __launch_bounds__(kThreads)
render_tiles_kernel(const __grid_constant__ CubeDesc c, const __grid_constant__ ViewDesc V,
                    const __grid_constant__ TFDesc T, const __grid_constant__ RenderArgs A,
                    const PartialDev* __restrict__ parts, int n_parts) {
    __shared__ float4 tab[256];
    __shared__ unsigned mask[kCullChunk / 32];
    if (MODE == VR_MODE_EA) load_tf(tab, T.baked);
    int tx, ty; tile_pixel(tx, ty);
    const int x0 = blockIdx.x * kTileW, y0 = blockIdx.y * kTileH;
    const int i = x0 + tx, j = y0 + ty;
    const bool live = i < V.W && j < V.H;
    Ray r; r.k0 = 0; r.k1 = -1;
    r.o[0] = r.o[1] = r.o[2] = 0.f; r.d[0] = r.d[1] = r.d[2] = 0.f; r.step = V.step; r.margin = 0.f;
    r.inv[0] = r.inv[1] = r.inv[2] = 0.f;
    if (live) setup_ray(V, c, i, j, r);
    Stats st = {0, 0, 0};
    unsigned long long nominal = 0, n_stopped = 0;
    for (int base = 0; base < n_parts; base += kCullChunk) {
        const int cnt = min(kCullChunk, n_parts - base);
        __syncthreads();
        if (threadIdx.x < kCullChunk / 32) mask[threadIdx.x] = 0u;
        __syncthreads();
        for (int q = threadIdx.x; q < cnt; q += kThreads) {
            const PartialDev& P = parts[base + q];
            if (P.x0 < x0 + kTileW && P.x0 + P.w > x0 && P.y0 < y0 + kTileH && P.y0 + P.h > y0) atomicOr(&mask[q >> 5], 1u << (q & 31));
        }
        __syncthreads();
        for (int w = 0; w < (cnt + 31) / 32; ++w) {
            for (unsigned bits = mask[w]; bits; bits &= bits - 1) {
                const PartialDev& P = parts[base + 32 * w + __ffs(bits) - 1];
                const int lx = i - P.x0, ly = j - P.y0;
                const bool mine = live && lx >= 0 && ly >= 0 && lx < P.w && ly < P.h;
                const int bid = P.brick;
                const int b[3] = {P.b[0], P.b[1], P.b[2]};
                const int lo[3] = {b[0] * c.B[0], b[1] * c.B[1], b[2] * c.B[2]};
                int ka = mine ? r.k0 : 0, kb = mine ? r.k1 : -1;
                brick_interval(c, r, b, lo, ka, kb);
                Accum acc = {{0.f, 0.f, 0.f}, 0.f, -INFINITY};
                const bool stopped = march_interval<MODE, LAYOUT, JUMP, VT>(c, r, T, A, tab, bid, lo, ka, kb, acc, st);
                if (mine) {
                    const long long px = (long long)ly * P.pitch + lx;
                    if (MODE == VR_MODE_MIP) reinterpret_cast<float*>(P.data)[px] = acc.m;
                    else reinterpret_cast<float4*>(P.data)[px] = make_float4(acc.C[0], acc.C[1], acc.C[2], acc.A);
                }
                if (kb >= ka) nominal += (unsigned long long)(kb - ka + 1);
                if (stopped) ++n_stopped;
            }
        }
    }
    if (A.counters) {
        count(A.counters, kNominal, nominal);
        count(A.counters, kTaken, st.taken);
        count(A.counters, kVisited, st.visit);
        count(A.counters, kSkipped, st.skip);
        count(A.counters, kTerminated, n_stopped);
    }
}

// ================================================================== variant 3: lockstep
// A warp owns the 32 rays of its 8 x 4 pixel tile and walks them TOGETHER through chunks of 32
// lattice indices [kbase, kbase + 31] (k counts from the near plane, so a chunk is a thin shell
// that all 32 rays cross at about the same place: lines shared by neighbouring rays are fetched
// once and hit in L1 / L2, not re-read from HBM).  Inside a chunk the rays are taken one after the
// other, SAMPLE-PARALLEL: the 32 lanes take the 32 samples of that ray in the chunk (positions,
// O-3; gathers and trilinear interpolation, O-4), so the lanes' addresses follow the ray.
//
// The gathers are asynchronous copies (cp.async, 4 bytes each) into a per-lane ring of kDepth
// slots in shared memory: the 8 voxels of the ray taken kDepth - 1 steps later are requested
// before the current ones are interpolated, they occupy no register and stall no scoreboard.
//
// The values are then folded in ray order (O-5 / O-7) by the lane that owns the ray, whose
// accumulator never leaves it, so early ray termination (O-7) is exact per ray:
//   MIP        - max is exact in any order: a warp reduction, then lane r takes the maximum;
//   EA, SPARSE - the few samples whose table coordinate is not below x_clear (see fold) are
//                handed to lane r one by one with a shuffle, in lattice order;
//   EA, DENSE  - the values go to shared memory, vals[ray][sample], and after the last ray of
//                the chunk every lane folds the 32 values of ITS ray front to back (all 32 rays
//                in parallel), so opaque transfer functions cost the same as sparse ones.
// Skipped samples (O-10) are never interpolated or folded.  All three give identical frames.
//
// REGS: the same ring in REGISTERS (plain loads, 3 rays ahead, 5 CTAs per SM).  The shared-memory side
// of a 4-byte cp.async takes one L1 wavefront per arriving sector; rays that run along z (the short
// axis of the 4 x 4 x 2 micro-blocks) meet the most sectors per request and are faster with plain
// loads (MIP on C3: 17.3 -> 14.7 ms), rays along x or y with cp.async (12.7 vs 14.1 ms): RenderArgs::ring.
constexpr int kValPitch = 33;
#ifndef VR_OCC_GROUP
#define VR_OCC_GROUP 8
#endif
#ifndef VR_OCC_CTAS
#define VR_OCC_CTAS 8
#endif
#ifndef VR_DEPTH_REGS
#define VR_DEPTH_REGS 3
#endif
#ifndef VR_DENSE_TEST
#define VR_DENSE_TEST 2
#endif
#ifndef VR_PIN_OCC0
#define VR_PIN_OCC0 1
#endif
#ifndef VR_DENSE_CTAS
#define VR_DENSE_CTAS 8
#endif
#ifndef VR_BEAM_COARSE
#define VR_BEAM_COARSE true
#endif
#ifndef VR_RUNS_GROUP
#define VR_RUNS_GROUP 4
#endif
#ifndef VR_REGS_CTAS
#define VR_REGS_CTAS 5
#endif
constexpr int kDepth = 3;               // rays in flight per warp (measured: 2 -> 12.1, 3 -> 12.0, 4 -> 13.5 ms on C3)
constexpr int kDepthRegs = VR_DEPTH_REGS;   // the same for the register ring
constexpr int kBitsWords = 1024;        // shared copy of one brick's macro-cell bits (256^3 bricks: 32^3 cells)

__device__ __forceinline__ void cp_async4(unsigned dst, const float* src) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(dst), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

// Request the 8 voxels of gather8 into dst[e * 32] (floats, e = 0..7; dst is a shared address in bytes).
template <int LAYOUT>
__device__ __forceinline__ void gather8_async(const BrickRef& b, int ix, int iy, int iz, unsigned dst) {
    unsigned q, dx, dy, dz;
    cell_address<LAYOUT>(b, (unsigned)(ix - b.lo[0]), (unsigned)(iy - b.lo[1]), (unsigned)(iz - b.lo[2]), q, dx, dy, dz);
    const float* p = b.base + q;
    cp_async4(dst, p);             cp_async4(dst + 128, p + dx);
    cp_async4(dst + 256, p + dy);  cp_async4(dst + 384, p + dy + dx);
    cp_async4(dst + 512, p + dz);  cp_async4(dst + 640, p + dz + dx);
    cp_async4(dst + 768, p + dz + dy); cp_async4(dst + 896, p + dz + dy + dx);
}

struct Slot { float w[3]; int rc; bool idle; float v[8]; };   // one ray in flight: weights of this lane's sample (v: register ring only)

// 7 CTAs per SM: 72 registers; an 8th CTA (64 registers) would shrink L1 to 28 KB and costs 10 % (measured)
template <int MODE, int LAYOUT, bool GLOBAL, bool DENSE, bool REGS, typename VT = float>
// register ring: 5 CTAs per SM for MIP; emission-absorption has its fold phase, in which a warp keeps no load in flight, and
// gains from a sixth CTA to cover it (C3 with a dense table 18.6 -> 17.5 ms; MIP is indifferent: 12.7 - 13.1 either way)
__global__ void __launch_bounds__(kThreads, REGS ? (MODE == VR_MODE_EA ? VR_REGS_CTAS + 1 : VR_REGS_CTAS) : 7)
render_ls_kernel(const __grid_constant__ CubeDesc c, const __grid_constant__ ViewDesc V,
                 const __grid_constant__ TFDesc T, const __grid_constant__ RenderArgs A,
                 const PartialDev* __restrict__ parts, int n_parts) {
    constexpr bool EA = MODE == VR_MODE_EA;
    constexpr bool VALS = EA && DENSE;
    constexpr bool SBITS = EA && !GLOBAL;
    constexpr int kWarps = kThreads / 32;
    __shared__ float4 tab[EA ? 256 : 1];
    __shared__ PartialDev part;
    __shared__ float4 rays_all[kWarps][64];
    constexpr int D = REGS ? kDepthRegs : kDepth;
    __shared__ float stage_all[REGS ? 1 : kWarps][REGS ? 1 : kDepth * 256];
    __shared__ float vals_all[VALS ? kWarps : 1][VALS ? 32 * kValPitch : 1];
    __shared__ unsigned sbits[SBITS ? kBitsWords : 1];
    int fx, fy;                                             // view pixel of this thread's ray
    bool live;
    if (GLOBAL) {
        int tx, ty; tile_pixel(tx, ty);
        fx = blockIdx.x * kTileW + tx; fy = blockIdx.y * kTileH + ty;
        live = fx < V.W && fy < V.H;
    } else {
        int lx, ly;
        live = locate_tile(parts, n_parts, part, lx, ly);
        fx = lx; fy = ly;
    }
    const bool cells = A.skip >= 2;
    int bid0 = 0, lo0[3] = {0, 0, 0};
    if (!GLOBAL) {
        bid0 = part.brick;
        lo0[0] = part.b[0] * c.B[0]; lo0[1] = part.b[1] * c.B[1]; lo0[2] = part.b[2] * c.B[2];
    }
    const bool bits_shared = SBITS && cells && c.cell_words_per_brick <= kBitsWords;
    if (bits_shared)
        for (int i = threadIdx.x; i < c.cell_words_per_brick; i += kThreads)
            sbits[i] = __ldg(&c.cell_bits[(long long)bid0 * c.cell_words_per_brick + i]);
    if (EA) load_tf(tab, T.baked);                          // ends with __syncthreads()
    Ray r; r.k0 = 0; r.k1 = -1;
    r.o[0] = r.o[1] = r.o[2] = 0.f; r.d[0] = r.d[1] = r.d[2] = 0.f; r.step = V.step; r.margin = 0.f;
    if (live) setup_ray(V, c, GLOBAL ? fx : part.x0 + fx, GLOBAL ? fy : part.y0 + fy, r);
    int ka = r.k0, kb = r.k1;
    if (!GLOBAL) {
        const int b[3] = {part.b[0], part.b[1], part.b[2]};
        brick_interval(c, r, b, lo0, ka, kb);
    }
    BrickRefT<VT> br0 = brick_ref<LAYOUT, VT>(c, bid0, lo0);
    if (!GLOBAL) asm volatile("" : "+l"(br0.base));         // the brick's base stays in two registers (else re-derived from the brick id per sample)
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    float* vals = vals_all[VALS ? warp : 0];
    float4* rays = rays_all[warp];
    const float* stage = stage_all[REGS ? 0 : warp] + (REGS ? 0 : lane);
    const unsigned stage_addr = (unsigned)__cvta_generic_to_shared(stage);
    rays[2 * lane] = make_float4(r.o[0], r.o[1], r.o[2], r.d[0]);
    rays[2 * lane + 1] = make_float4(r.d[1], r.d[2], __int_as_float(ka), __int_as_float(kb));
    __syncwarp();
    bool alive = ka <= kb, stopped = false;
    int k_end = kb;                                         // last lattice index this ray got to (ERT: the stop)
    int K0 = alive ? ka : 0x7fffffff, K1 = alive ? kb : -1;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        K0 = min(K0, __shfl_xor_sync(0xffffffffu, K0, o));
        K1 = max(K1, __shfl_xor_sync(0xffffffffu, K1, o));
    }
    Accum acc = {{0.f, 0.f, 0.f}, 0.f, -INFINITY};
    unsigned n_taken = 0;
    // sort-last MIP: once a ray's maximum has reached the brick's maximum nothing in the brick can raise it (O-10 at the
    // brick level, exact; an all-zero brick of flagged channels is left after its first chunk)
    const float brick_max = (!EA && !GLOBAL && A.skip >= 1) ? __ldg(&c.brick_mm[bid0]).y : INFINITY;
    for (int kbase = K0; kbase <= K1; kbase += 32) {
        if (!EA && !GLOBAL && brick_max <= acc.m) alive = false;
        if (!__ballot_sync(0xffffffffu, alive)) break;
        const unsigned act = __ballot_sync(0xffffffffu, alive && ka <= kbase + 31 && kb >= kbase);
        if (!act) continue;
        const int k = kbase + lane;                         // this lane's sample of every ray of the chunk
        const float t = __fmul_rn((float)k, r.step);        // O-3: t_k = k * Delta
        unsigned rest = act;
        // request the 8 voxels of this lane's sample of the next ray of the chunk (if any) into slot s
        auto issue = [&](Slot& S, const int s) {
            S.rc = -1; S.idle = true;
            S.w[0] = S.w[1] = S.w[2] = 0.f;
            if (REGS) {
#pragma unroll
                for (int e = 0; e < 8; ++e) S.v[e] = 0.f;
            }
            if (rest) {
                const int rr = __ffs(rest) - 1;
                rest &= rest - 1;
                S.rc = rr;
                const float4 ra = rays[2 * rr], rb = rays[2 * rr + 1];
                float m_r = -INFINITY;
                if (!EA) m_r = __shfl_sync(0xffffffffu, acc.m, rr);
                if (k >= __float_as_int(rb.z) && k <= __float_as_int(rb.w)) {
                    float p[3], fl[3];
                    p[0] = __fmaf_rn(t, ra.w, ra.x); p[1] = __fmaf_rn(t, rb.x, ra.y); p[2] = __fmaf_rn(t, rb.y, ra.z);
                    const int iv[3] = {floor_pos(p[0], fl[0]), floor_pos(p[1], fl[1]), floor_pos(p[2], fl[2])};
                    S.w[0] = __fsub_rn(p[0], fl[0]); S.w[1] = __fsub_rn(p[1], fl[1]); S.w[2] = __fsub_rn(p[2], fl[2]);
                    if (GLOBAL) {
                        int b[3]; brick_of(c, iv, b);
                        const int lo[3] = {b[0] * c.B[0], b[1] * c.B[1], b[2] * c.B[2]};
                        const int bid = b[0] + c.G[0] * (b[1] + c.G[1] * b[2]);
                        bool idle = false;
                        if (A.skip) {                       // O-10 (exact), per sample
                            if (!EA) idle = __ldg(&c.brick_mm[bid]).y <= m_r;
                            else idle = __ldg(&c.brick_active[bid]) == 0;
                            if (cells && !idle) idle = cell_idle<MODE>(c, bid, lo, iv[0], iv[1], iv[2], m_r);
                        }
                        S.idle = idle;
                        if (!idle) {
                            if constexpr (REGS) gather8<LAYOUT>(brick_ref<LAYOUT, VT>(c, bid, lo), iv[0], iv[1], iv[2], S.v);
                            else gather8_async<LAYOUT>(brick_ref<LAYOUT, VT>(c, bid, lo), iv[0], iv[1], iv[2], stage_addr + 1024u * s);
                        }
                    } else {
                        bool idle = false;
                        if (bits_shared) {
                            const int cidx = ((iv[0] - lo0[0]) >> 3) + c.C[0] * (((iv[1] - lo0[1]) >> 3) + c.C[1] * ((iv[2] - lo0[2]) >> 3));
                            idle = ((sbits[cidx >> 5] >> (cidx & 31)) & 1u) == 0u;
                        } else if (cells) idle = cell_idle<MODE>(c, bid0, lo0, iv[0], iv[1], iv[2], m_r);
                        S.idle = idle;
                        if (!idle) {
                            if constexpr (REGS) gather8<LAYOUT>(br0, iv[0], iv[1], iv[2], S.v);
                            else gather8_async<LAYOUT>(br0, iv[0], iv[1], iv[2], stage_addr + 1024u * s);
                        }
                    }
                }
            }
            cp_async_commit();
        };
        unsigned my_fold = 0u, my_done = 0u;                // DENSE: this lane's ray: samples to fold / interpolated
        // interpolate the samples of the ray in slot s (its copies have landed) and fold them
        auto consume = [&](const Slot& S, const int s) {
            float v[8];
            if (REGS) {
#pragma unroll
                for (int e = 0; e < 8; ++e) v[e] = S.v[e];
            } else {
                const float* st = stage + 256 * s;
#pragma unroll
                for (int e = 0; e < 8; ++e) v[e] = st[32 * e];
            }
            const float val = trilinear(v, S.w[0], S.w[1], S.w[2]);       // idle lanes: stale values, never used
            const unsigned done_bits = __ballot_sync(0xffffffffu, !S.idle);
            if (!EA) {
                // warp maximum by one redux.sync on a key that orders floats as integers (no NaN here: refused at upload)
                const int bits = __float_as_int(S.idle ? -INFINITY : val);
                const int top = __reduce_max_sync(0xffffffffu, bits ^ ((bits >> 31) & 0x7fffffff));
                const float m = __int_as_float(top ^ ((top >> 31) & 0x7fffffff));
                if (lane == S.rc) { acc.m = fmaxf(acc.m, m); n_taken += __popc(done_bits); }
                return;
            }
            // samples whose table coordinate lies below x_clear have weight exactly zero (see fold)
            const bool need = !S.idle && !(__fmul_rn(__fsub_rn(val, T.vmin), T.scale) < T.x_clear);
            const unsigned fold_bits = __ballot_sync(0xffffffffu, need);
            if (VALS) {
                vals[S.rc * kValPitch + lane] = val;
                if (lane == S.rc) { my_fold = fold_bits; my_done = done_bits; }
                return;
            }
            unsigned upto = 0xffffffffu;
            for (unsigned bits = fold_bits; bits; bits &= bits - 1) {
                const int l = __ffs(bits) - 1;
                const float vl = __shfl_sync(0xffffffffu, val, l);
                if (lane == S.rc && alive && fold<MODE>(acc, vl, tab, T, A.tau)) {
                    stopped = true; alive = false; k_end = kbase + l;
                    upto = l >= 31 ? 0xffffffffu : ((1u << (l + 1)) - 1u);
                }
            }
            if (lane == S.rc) n_taken += __popc(done_bits & upto);
        };
        Slot slot[D];
#pragma unroll
        for (int s = 0; s < D - 1; ++s) issue(slot[s], s);
        for (bool more = true; more;) {
#pragma unroll
            for (int u = 0; u < D; ++u) {
                issue(slot[(u + D - 1) % D], (u + D - 1) % D);
                cp_async_wait<D - 1>();
                if (slot[u].rc < 0) { more = false; break; }
                consume(slot[u], u);
            }
        }
        if (VALS) {
            __syncwarp();
            // lane = ray: fold its flagged values front to back
            if ((act >> lane) & 1u) {
                const float* mine = vals + lane * kValPitch;
                unsigned upto = 0xffffffffu;
                for (unsigned bits = my_fold; bits; bits &= bits - 1) {
                    const int l = __ffs(bits) - 1;
                    if (fold<MODE>(acc, mine[l], tab, T, A.tau)) {
                        stopped = true; alive = false; k_end = kbase + l;
                        upto = l >= 31 ? 0xffffffffu : ((1u << (l + 1)) - 1u);
                        break;
                    }
                }
                n_taken += __popc(my_done & upto);
            }
            __syncwarp();
        }
    }
    if (live) {
        if (GLOBAL) write_frame_pixel<MODE>(V, T, A, fx, fy, acc, r.k1 >= r.k0);
        else {
            const long long px = (long long)fy * part.pitch + fx;
            if (!EA) reinterpret_cast<float*>(part.data)[px] = acc.m;
            else reinterpret_cast<float4*>(part.data)[px] = make_float4(acc.C[0], acc.C[1], acc.C[2], acc.A);
        }
    }
    if (A.counters) {
        const unsigned long long nom = kb >= ka ? (unsigned long long)(kb - ka + 1) : 0ULL;
        const unsigned long long reached = kb >= ka ? (unsigned long long)(k_end - ka + 1) : 0ULL;
        if (GLOBAL) count(A.counters, kRays, nom ? 1 : 0);
        count(A.counters, kNominal, nom);
        count(A.counters, kTaken, n_taken);
        count(A.counters, kVisited, nom ? 1 : 0);
        count(A.counters, kSkipped, reached - n_taken);     // lattice samples passed over by O-10
        count(A.counters, kTerminated, stopped ? 1 : 0);
    }
}

// ================================================================== variant 3 for sparse tables: test, compact, gather, fold
// Same ownership as render_ls_kernel (a warp walks its 32 rays together through chunks of 32
// lattice indices), but a sample is first TESTED against the occupancy bits (CubeDesc::occ, O-10
// at the level of one trilinear cell): only samples whose 8 corners can reach a table entry of
// non-zero opacity are interpolated.  Per chunk:
//   test   - lane = ray: every lane walks the 32 lattice indices of the chunk along ITS ray and
//            looks up the bit of each sample (position and floor only; the next sample's word is
//            requested before the current one is tested) -> one 32-bit mask per ray;
//   list   - the survivors of all rays are written to a list in shared memory, ray-major, lattice
//            order inside a ray (warp prefix sum of the masks' populations);
//   gather - lane = list entry, 32 entries per step (full lanes however few samples survive):
//            position and weights are recomputed (the same float32 operations), the 8 voxels come
//            through the cp.async ring, the value goes to vals[list index];
//   fold   - lane = ray: the owner folds its entries front to back (O-7, exact ERT).
// A list longer than kListCap is taken in batches of whole rays (dense tables use
// render_ls_kernel<..., DENSE> instead).  Frames are identical to the other marchers': a skipped
// sample has weight exactly zero.
#ifndef VR_LIST_CAP
#define VR_LIST_CAP 256
#endif
#ifndef VR_DENSE_LIST_CAP
#define VR_DENSE_LIST_CAP 512
#endif
// entries per batch.  Sparse rays (C3) live on L1: more shared memory per CTA costs more than the batches save (256 -> 512:
// 5.4 -> 13.7 ms); dense rays meet whole sources, where every sample survives, and gain from longer batches (C4 19.6 ->
// 18.8, C5 52.9 -> 50.3 ms)
template <int TEST> constexpr int kListCapOf = TEST == 0 ? VR_LIST_CAP : VR_DENSE_LIST_CAP;
constexpr int kOccDepth = 2;             // gathers are few here: a shallower ring leaves more of the SM to L1 (3 -> 6.36, 2 -> 6.26 ms)

// 8 CTAs per SM (64 registers): the few gathers leave L1 alone, more warps hide the bit lookups (measured:
// 7 -> 6.83, 8 -> 6.44, 9 -> 7.27 ms on C3)
template <bool GLOBAL, typename VT = float, bool ASYNC = true, int TEST = 0>
__global__ void __launch_bounds__(kThreads, ASYNC ? (TEST == 2 ? VR_DENSE_CTAS : VR_OCC_CTAS) : 6)      // gathers held in registers: 80 instead of 64
render_occ_kernel(const __grid_constant__ CubeDesc c, const __grid_constant__ ViewDesc V,
                  const __grid_constant__ TFDesc T, const __grid_constant__ RenderArgs A,
                  const PartialDev* __restrict__ parts, int n_parts) {
    constexpr int MODE = VR_MODE_EA, LAYOUT = 1;
    constexpr int kWarps = kThreads / 32;
    constexpr int kListCap = kListCapOf<TEST>;
    __shared__ float4 rays_all[kWarps][64];
    __shared__ float stage_all[ASYNC ? kWarps : 1][ASYNC ? kOccDepth * 256 : 1];
    __shared__ float vals_all[kWarps][kListCap];
    __shared__ unsigned short list_all[kWarps][kListCap];
    __shared__ unsigned mask[GLOBAL ? 1 : kCullChunk / 32];
    // one CTA per pixel tile of the view; for partial images it walks every brick over the tile, so
    // the ray is set up once (fp64) per pixel, not once per (pixel, brick)
    int tx, ty; tile_pixel(tx, ty);
    const int x0 = blockIdx.x * kTileW, y0 = blockIdx.y * kTileH;
    const int fx = x0 + tx, fy = y0 + ty;
    const bool live = fx < V.W && fy < V.H;
    Ray r; r.k0 = 0; r.k1 = -1;
    r.o[0] = r.o[1] = r.o[2] = 0.f; r.d[0] = r.d[1] = r.d[2] = 0.f; r.step = V.step; r.margin = 0.f;
    if (live) setup_ray(V, c, fx, fy, r);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    float* vals = vals_all[warp];
    unsigned short* list = list_all[warp];
    float4* rays = rays_all[warp];
    const float* stage = stage_all[ASYNC ? warp : 0] + (ASYNC ? lane : 0);
    const unsigned stage_addr = (unsigned)__cvta_generic_to_shared(stage);
    rays[2 * lane] = make_float4(r.o[0], r.o[1], r.o[2], r.d[0]);
    // state of the brick being marched (GLOBAL: the whole cube in one go)
    int bid0 = 0, lo0[3] = {0, 0, 0};
    BrickRefT<VT> br0 = brick_ref<LAYOUT, VT>(c, 0, lo0);
    const unsigned* occ0 = c.occ;
    const unsigned* cbits0 = c.cell_bits;
    int ka = r.k0, kb = r.k1, k_end = kb;
    bool alive = false, stopped = false;
    Accum acc = {{0.f, 0.f, 0.f}, 0.f, -INFINITY};
    unsigned n_taken = 0;
    // the occupancy word of a sample (0 if its brick is inactive) and the sample's bit in it; 64-bit
    // brick offsets: a sharded cube's global brick ids times the words per brick can pass 2^32
    // `valid` false: the sample lies outside this lane's interval - the address arithmetic runs anyway (it cannot fault),
    // only the load is predicated: no branch around the ~25 instructions of a test (non-GLOBAL; 5 of ~30 were the branch)
    auto locate = [&](const float tk, unsigned& word, unsigned& bit, const bool valid = true) {
        float fl;
        const int iv[3] = {floor_pos(__fmaf_rn(tk, r.d[0], r.o[0]), fl), floor_pos(__fmaf_rn(tk, r.d[1], r.o[1]), fl),
                           floor_pos(__fmaf_rn(tk, r.d[2], r.o[2]), fl)};
        unsigned lx, ly, lz;
        const unsigned* occb;
        if (GLOBAL) {
            int b[3]; brick_of(c, iv, b);
            const int bid = b[0] + c.G[0] * (b[1] + c.G[1] * b[2]);
            lx = (unsigned)(iv[0] - b[0] * c.B[0]); ly = (unsigned)(iv[1] - b[1] * c.B[1]); lz = (unsigned)(iv[2] - b[2] * c.B[2]);
            occb = c.occ + (long long)bid * c.occ_words_per_brick;
            if (__ldg(&c.brick_active[bid]) == 0) { word = 0u; bit = 0u; return; }
        } else {
            lx = (unsigned)(iv[0] - lo0[0]); ly = (unsigned)(iv[1] - lo0[1]); lz = (unsigned)(iv[2] - lo0[2]);
            occb = occ0;
        }
        word = 0u;
        if (valid) word = __ldg(occb + occ_word_index(c, lx, ly, lz));   // an L1 hit while the ray stays in its 4 x 4 x 2 cells
        bit = occ_bit_index(lx, ly, lz);
    };
    // march the taken samples [ka, kb] of every lane's ray (all members of brick bid0 unless GLOBAL) into acc
    auto march = [&]() {
    rays[2 * lane + 1] = make_float4(r.d[1], r.d[2], __int_as_float(ka), __int_as_float(kb));
    __syncwarp();
    alive = ka <= kb; stopped = false; k_end = kb; n_taken = 0;
    acc.C[0] = acc.C[1] = acc.C[2] = 0.f; acc.A = 0.f; acc.m = -INFINITY;
    const int K0 = __reduce_min_sync(0xffffffffu, alive ? ka : 0x7fffffff), K1 = __reduce_max_sync(0xffffffffu, alive ? kb : -1);
    int cur = ka, run_left = 0;                             // TEST 1: next lattice index to classify, rest of its macro-cell run
    bool run_on = false;
    unsigned beam_flags = 0u;                               // TEST 2: chunks of the current group of 4 whose beam meets a non-zero word
    // TEST 2: local voxel coordinates of the trilinear cell of this lane's sample k, k clipped to [klo, khi]
    auto cell_of = [&](int k, int klo, int khi, int l[3]) {
        const float tk = __fmul_rn((float)min(max(k, klo), khi), r.step);
        float fl;
        l[0] = floor_pos(__fmaf_rn(tk, r.d[0], r.o[0]), fl) - lo0[0];
        l[1] = floor_pos(__fmaf_rn(tk, r.d[1], r.o[1]), fl) - lo0[1];
        l[2] = floor_pos(__fmaf_rn(tk, r.d[2], r.o[2]), fl) - lo0[2];
    };
    // TEST 2: the beam against the occupancy words over four consecutive stretches of `stride` lattice indices from k0.
    // Stretch i holds every lane's samples k0 + i stride .. k0 + (i + 1) stride (one more than its share: conservative),
    // clipped to the lane's interval; positions are monotone along a ray, so the box of the two end samples holds the ones
    // between, and the box over the lanes (redux) holds the whole beam.  The 4 x 4 x 2 blocks of cells that meet box i are
    // shared out among lanes 8 i .. 8 i + 7, one occupancy word each per round, so the four stretches' loads are in flight
    // together.  Returns bit i = some word of stretch i is non-zero (warp-uniform).  One small loop: this is all a warp
    // runs while its beam crosses empty space.
    auto test4 = [&](const int k0, const int stride, const bool coarse) {
        const int grp = lane >> 3;
        int bl[3] = {0, 0, 0}, bh[3] = {-1, -1, -1}, ca[3], cb[3];
        cell_of(k0, ka, kb, ca);
#pragma unroll 1                                            // rolled: the loop a warp runs through empty space has to stay in the L0 instruction cache
        for (int i = 0; i < 4; ++i) {
            cell_of(k0 + stride * (i + 1), ka, kb, cb);
            const bool part = alive && ka <= k0 + stride * (i + 1) - 1 && kb >= k0 + stride * i;
#pragma unroll
            for (int x = 0; x < 3; ++x) {
                const int lo = __reduce_min_sync(0xffffffffu, part ? min(ca[x], cb[x]) : 0x7fffffff);
                const int hi = __reduce_max_sync(0xffffffffu, part ? max(ca[x], cb[x]) : -1);
                if (grp == i) { bl[x] = lo; bh[x] = hi; }
                ca[x] = cb[x];
            }
        }
        // coarse: the 8^3 macro-cells that meet the box (one activity bit each); else its 4 x 4 x 2 blocks (one word each)
        const int sx = coarse ? 3 : 2, sz = coarse ? 3 : 1;
        const int bx0 = bl[0] >> sx, by0 = bl[1] >> sx, bz0 = bl[2] >> sz;
        const int nx = (bh[0] >> sx) - bx0 + 1, ny = (bh[1] >> sx) - by0 + 1, nz = (bh[2] >> sz) - bz0 + 1;
        const int nxy = nx * ny, total = (nx > 0 && ny > 0 && nz > 0) ? nxy * nz : 0;
        const unsigned s0 = coarse ? (unsigned)c.C[0] : (unsigned)c.T[0], s1 = coarse ? (unsigned)c.C[1] : (unsigned)c.T[1];
        bool any = total > 2048;                            // an absurd box: not tested, taken as met
        if (!any) {
            const float rx = __frcp_rn((float)nx), rxy = __frcp_rn((float)nxy);
            for (int e = lane & 7; e < total; e += 8) {     // e -> (ex, ey, ez): (e + 1/2) / n floors exactly for these small integers
                const int ez = __float2int_rz(__fmul_rn((float)e + 0.5f, rxy)), rem = e - ez * nxy;
                const int ey = __float2int_rz(__fmul_rn((float)rem + 0.5f, rx)), ex = rem - ey * nx;
                const unsigned idx = (unsigned)(bx0 + ex) + s0 * ((unsigned)(by0 + ey) + s1 * (unsigned)(bz0 + ez));
                if (coarse) any |= ((__ldg(cbits0 + (idx >> 5)) >> (idx & 31u)) & 1u) != 0u;
                else any |= __ldg(occ0 + idx) != 0u;
            }
        }
        const unsigned v = __ballot_sync(0xffffffffu, any);
        return ((v & 0xffu) ? 1u : 0u) | ((v & 0xff00u) ? 2u : 0u) | ((v & 0xff0000u) ? 4u : 0u) | ((v & 0xff000000u) ? 8u : 0u);
    };
    for (int kbase = K0; kbase <= K1; kbase += 32) {
        if constexpr (TEST == 2) {
            const int sub = ((kbase - K0) >> 5) & 3;
            if (sub == 0) {                                 // four chunks at a time
                if (!__ballot_sync(0xffffffffu, alive)) break;
                beam_flags = test4(kbase, 32, VR_BEAM_COARSE);
                if (beam_flags == 0u) { kbase += 96; continue; }
            }
            if (((beam_flags >> sub) & 1u) == 0u) continue;
        }
        if (!__ballot_sync(0xffffffffu, alive)) break;
        const bool mine = alive && ka <= kbase + 31 && kb >= kbase;
        const unsigned act = __ballot_sync(0xffffffffu, mine);
        if (!act) continue;
        // ---- test, lane = ray: bit j of my_act <=> sample kbase + j of this lane's ray survives.  The
        // word of the next sample is requested before the current one is tested (reloading it every
        // time measured faster than keeping it in a register while the ray stays in its cells).
        unsigned my_act = 0u;
        if constexpr (TEST != 0) {
            // DENSE RAYS (neighbouring rays closer than a voxel).  The warp's 32 rays form a thin beam; `cand` = the samples
            // that go to the per-sample occupancy test, found per chunk in one of two ways:
            //  TEST 2 (partial images): the beam is tested as a whole against the occupancy WORDS (one per 4 x 4 x 2 block
            //   of cells): the bounding box of all 32 rays' samples of the chunk (positions are monotone along a ray, so
            //   the box of the samples at the two ends of every lane's part of the chunk), one block per lane; if every word
            //   is zero the chunk is left by the whole warp.  Otherwise the same test per quarter of the chunk (8 lattice
            //   indices); the samples of the quarters with a non-zero word are the candidates.  No per-ray traversal.
            //  TEST 1 (whole frame, O-8 GLOBAL): every lane cuts ITS part of the chunk into runs inside 8^3 macro-cells
            //   (one position, one run length and one activity bit per run; a run that leaves the chunk is carried into
            //   the next); the candidates are the samples of active runs.
            // Then the warp walks the candidate indices together, each lane looking up the occupancy bit of its own
            // sample at that index: the loop is uniform, so the lanes stay together whatever their rays skip (a ray
            // per thread that tests and samples on its own ran at a quarter of the lanes inside active cells).
            unsigned cand = 0u;
            if constexpr (TEST == 2) {
                // the chunk's beam met a non-zero word: the same test per quarter of the chunk; the samples of the quarters
                // that meet one are the candidates
                const unsigned q4 = test4(kbase, 8, false);
                const unsigned quarters = ((q4 & 1u) ? 0xffu : 0u) | ((q4 & 2u) ? 0xff00u : 0u) | ((q4 & 4u) ? 0xff0000u : 0u) | ((q4 & 8u) ? 0xff000000u : 0u);
                if (mine) cand = quarters & (0xffffffffu << (max(ka, kbase) - kbase)) & (0xffffffffu >> (31 - (min(kb, kbase + 31) - kbase)));
            } else if (mine) {
                const int kend = min(kb, kbase + 31);
                const int S8[3] = {kCell, kCell, kCell};
                while (cur <= kend) {
                    if (run_left == 0) {
                        float p[3], fl;
                        position(r, (float)cur, p);
                        const int iv[3] = {floor_pos(p[0], fl), floor_pos(p[1], fl), floor_pos(p[2], fl)};
                        int bid = bid0, lo[3] = {lo0[0], lo0[1], lo0[2]};
                        bool brick_on = true;
                        if (GLOBAL) {
                            int b[3]; brick_of(c, iv, b);
                            lo[0] = b[0] * c.B[0]; lo[1] = b[1] * c.B[1]; lo[2] = b[2] * c.B[2];
                            bid = b[0] + c.G[0] * (b[1] + c.G[1] * b[2]);
                            brick_on = __ldg(&c.brick_active[bid]) != 0;
                        }
                        if (brick_on) {
                            const int clo[3] = {lo[0] + (((iv[0] - lo[0]) >> 3) << 3), lo[1] + (((iv[1] - lo[1]) >> 3) << 3),
                                                lo[2] + (((iv[2] - lo[2]) >> 3) << 3)};
                            run_left = min(kb - cur + 1, run_length(r, p, clo, S8));
                            run_on = !cell_idle<MODE>(c, bid, lo, iv[0], iv[1], iv[2], 0.f);
                        } else {
                            run_left = min(kb - cur + 1, run_length(r, p, lo, c.B));
                            run_on = false;
                        }
                    }
                    const int take = min(run_left, kend - cur + 1);
                    if (run_on) cand |= (take >= 32 ? 0xffffffffu : ((1u << take) - 1u)) << (cur - kbase);
                    cur += take; run_left -= take;
                }
            }
            const unsigned all = __reduce_or_sync(0xffffffffu, cand);
            if (all == 0u) continue;
            for (unsigned bits = all; bits;) {
                int jj[VR_RUNS_GROUP];
                unsigned word[VR_RUNS_GROUP], bit[VR_RUNS_GROUP];
#pragma unroll
                for (int u = 0; u < VR_RUNS_GROUP; ++u) { jj[u] = bits ? __ffs(bits) - 1 : -1; bits &= bits - 1; }
#pragma unroll
                for (int u = 0; u < VR_RUNS_GROUP; ++u) {
                    if constexpr (GLOBAL) {
                        word[u] = 0u; bit[u] = 0u;
                        if (jj[u] >= 0 && ((cand >> jj[u]) & 1u)) locate(__fmul_rn((float)(kbase + jj[u]), r.step), word[u], bit[u]);
                    } else locate(__fmul_rn((float)(kbase + max(jj[u], 0)), r.step), word[u], bit[u], jj[u] >= 0 && ((cand >> (jj[u] & 31)) & 1u));
                }
#pragma unroll
                for (int u = 0; u < VR_RUNS_GROUP; ++u) my_act |= ((word[u] >> bit[u]) & 1u) << (jj[u] & 31);
            }
        } else {
            int j0 = mine ? max(ka, kbase) - kbase : 32, j1 = mine ? min(kb, kbase + 31) - kbase : -1;
            const int J0 = __reduce_min_sync(0xffffffffu, j0), J1 = __reduce_max_sync(0xffffffffu, j1);
#if VR_OCC_GROUP <= 1
            unsigned word = 0u, bit = 0u;                            // of sample j
            if (J0 >= j0 && J0 <= j1) locate(__fmul_rn((float)(kbase + J0), r.step), word, bit);
            for (int j = J0; j <= J1; ++j) {
                unsigned nword = 0u, nbit = 0u;                      // of sample j + 1
                if (j + 1 >= j0 && j + 1 <= j1) locate(__fmul_rn((float)(kbase + j + 1), r.step), nword, nbit);
                if (j >= j0 && j <= j1 && ((word >> bit) & 1u)) my_act |= 1u << j;
                word = nword; bit = nbit;
            }
#else
            // VR_OCC_GROUP words are requested before the first of them is tested: with one request ahead the warp
            // waited on the word at its use (ncu: 45 % of the kernel's stall samples on that one shift)
            for (int j = J0; j <= J1; j += VR_OCC_GROUP) {
                unsigned word[VR_OCC_GROUP], bit[VR_OCC_GROUP];
#pragma unroll
                for (int u = 0; u < VR_OCC_GROUP; ++u) {
                    if constexpr (GLOBAL) {
                        word[u] = 0u; bit[u] = 0u;                   // out of this ray's range: reads as idle
                        if (j + u >= j0 && j + u <= j1) locate(__fmul_rn((float)(kbase + j + u), r.step), word[u], bit[u]);
                    } else locate(__fmul_rn((float)(kbase + j + u), r.step), word[u], bit[u], j + u >= j0 && j + u <= j1);
                }
#pragma unroll
                for (int u = 0; u < VR_OCC_GROUP; ++u) my_act |= ((word[u] >> bit[u]) & 1u) << ((j + u) & 31);
            }
#endif
        }
        // ---- list, ray-major: lane's entries at [off, off + cnt)
        const int cnt = __popc(my_act);
        int incl = cnt;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int up = __shfl_up_sync(0xffffffffu, incl, o);
            if (lane >= o) incl += up;
        }
        const int off = incl - cnt, total = __shfl_sync(0xffffffffu, incl, 31);
        for (int base = 0; base < total;) {                 // batches of whole rays, at most kListCap entries
            const bool inb = cnt > 0 && off >= base && off + cnt <= base + kListCap;
            const unsigned bm = __ballot_sync(0xffffffffu, inb);
            const int bend = __shfl_sync(0xffffffffu, off + cnt, 31 - __clz((int)bm));
            const int ntot = bend - base, my_start = off - base;
            if (inb) {
                int i = my_start;
                for (unsigned bits = my_act; bits; bits &= bits - 1) list[i++] = (unsigned short)((lane << 5) | (__ffs(bits) - 1));
            }
            __syncwarp();
            // ---- gather: one list entry per lane, 32 entries per step, through the cp.async ring
            const int ngroups = (ntot + 31) >> 5;
            auto issue = [&](Slot& S, const int g, const int s) {
                S.rc = g < ngroups ? g : -1; S.idle = true;
                S.w[0] = S.w[1] = S.w[2] = 0.f;
                const int idx = 32 * g + lane;
                if (g < ngroups && idx < ntot) {
                    const unsigned e = list[idx];
                    const int rr = (int)(e >> 5);
                    const float tt = __fmul_rn((float)(kbase + (int)(e & 31u)), r.step);
                    const float4 ra = rays[2 * rr], rb = rays[2 * rr + 1];
                    float p[3], fl[3];
                    p[0] = __fmaf_rn(tt, ra.w, ra.x); p[1] = __fmaf_rn(tt, rb.x, ra.y); p[2] = __fmaf_rn(tt, rb.y, ra.z);
                    const int iv[3] = {floor_pos(p[0], fl[0]), floor_pos(p[1], fl[1]), floor_pos(p[2], fl[2])};
                    S.w[0] = __fsub_rn(p[0], fl[0]); S.w[1] = __fsub_rn(p[1], fl[1]); S.w[2] = __fsub_rn(p[2], fl[2]);
                    S.idle = false;
                    if (GLOBAL) {
                        int b[3]; brick_of(c, iv, b);
                        const int lo[3] = {b[0] * c.B[0], b[1] * c.B[1], b[2] * c.B[2]};
                        const int bid = b[0] + c.G[0] * (b[1] + c.G[1] * b[2]);
                        if constexpr (ASYNC) gather8_async<LAYOUT>(brick_ref<LAYOUT, VT>(c, bid, lo), iv[0], iv[1], iv[2], stage_addr + 1024u * s);
                        else gather8<LAYOUT>(brick_ref<LAYOUT, VT>(c, bid, lo), iv[0], iv[1], iv[2], S.v);
                    } else {
                        if constexpr (ASYNC) gather8_async<LAYOUT>(br0, iv[0], iv[1], iv[2], stage_addr + 1024u * s);
                        else gather8<LAYOUT>(br0, iv[0], iv[1], iv[2], S.v);
                    }
                }
                cp_async_commit();
            };
            auto consume = [&](const Slot& S, const int s) {
                if (S.idle) return;
                float v[8];
                if constexpr (ASYNC) {
                    const float* st = stage + 256 * s;
#pragma unroll
                    for (int e = 0; e < 8; ++e) v[e] = st[32 * e];
                } else {
#pragma unroll
                    for (int e = 0; e < 8; ++e) v[e] = S.v[e];
                }
                vals[32 * S.rc + lane] = trilinear(v, S.w[0], S.w[1], S.w[2]);
            };
            Slot slot[kOccDepth];
            int gi = 0;
#pragma unroll
            for (int s = 0; s < kOccDepth - 1; ++s) issue(slot[s], gi++, s);
            for (bool more = true; more;) {
#pragma unroll
                for (int u = 0; u < kOccDepth; ++u) {
                    issue(slot[(u + kOccDepth - 1) % kOccDepth], gi++, (u + kOccDepth - 1) % kOccDepth);
                    cp_async_wait<kOccDepth - 1>();
                    if (slot[u].rc < 0) { more = false; break; }
                    consume(slot[u], u);
                }
            }
            __syncwarp();
            // ---- fold: lane = ray, its entries front to back (O-7).  (Looking the colours up first, with lane = list entry
            // and full lanes, and folding (r, g, b, a') from shared memory cost more shared memory than it saved: -3 %.)
            if (inb) {
                int i = 0;
                while (i < cnt) {
                    const bool stop = fold<MODE>(acc, vals[my_start + i], T.baked, T, A.tau);
                    ++i;
                    if (stop) { stopped = true; alive = false; k_end = kbase + (int)(list[my_start + i - 1] & 31u); break; }
                }
                n_taken += (unsigned)i;
            }
            __syncwarp();
            base = bend;
        }
    }
    __syncwarp();
    };
    unsigned long long c_nom = 0, c_reached = 0, c_taken = 0, c_stopped = 0;
    auto tally = [&]() {
        if (kb >= ka) { c_nom += (unsigned long long)(kb - ka + 1); c_reached += (unsigned long long)(k_end - ka + 1); }
        c_taken += n_taken;
        if (stopped) ++c_stopped;
    };
    if (GLOBAL) {
        march();
        tally();
        if (live) write_frame_pixel<MODE>(V, T, A, fx, fy, acc, r.k1 >= r.k0);
    } else {
        for (int base = 0; base < n_parts; base += kCullChunk) {
            const int cnt = min(kCullChunk, n_parts - base);
            __syncthreads();
            if (threadIdx.x < kCullChunk / 32) mask[threadIdx.x] = 0u;
            __syncthreads();
            for (int q = threadIdx.x; q < cnt; q += kThreads) {
                const PartialDev& P = parts[base + q];
                if (P.x0 < x0 + kTileW && P.x0 + P.w > x0 && P.y0 < y0 + kTileH && P.y0 + P.h > y0) atomicOr(&mask[q >> 5], 1u << (q & 31));
            }
            __syncthreads();
            for (int w = 0; w < (cnt + 31) / 32; ++w) {
                for (unsigned bits = mask[w]; bits; bits &= bits - 1) {
                    const PartialDev& P = parts[base + 32 * w + __ffs(bits) - 1];
                    const int lx = fx - P.x0, ly = fy - P.y0;
                    const bool mine = live && lx >= 0 && ly >= 0 && lx < P.w && ly < P.h;
                    bid0 = P.brick;
                    const int b[3] = {P.b[0], P.b[1], P.b[2]};
                    lo0[0] = b[0] * c.B[0]; lo0[1] = b[1] * c.B[1]; lo0[2] = b[2] * c.B[2];
                    br0 = brick_ref<LAYOUT, VT>(c, bid0, lo0);
#if VR_PIN_OCC0
                    asm volatile("" : "+l"(br0.base));
#endif
                    occ0 = c.occ + (long long)bid0 * c.occ_words_per_brick;
#if VR_PIN_OCC0
                    asm volatile("" : "+l"(occ0));          // kept in two registers: otherwise re-derived from the brick id at every sample (3 instructions of ~33)
#endif
                    cbits0 = c.cell_bits + (long long)bid0 * c.cell_words_per_brick;
#if VR_PIN_OCC0
                    if constexpr (TEST == 2) asm volatile("" : "+l"(cbits0));
#endif
                    ka = mine ? r.k0 : 0; kb = mine ? r.k1 : -1;
                    brick_interval(c, r, b, lo0, ka, kb);
                    march();
                    tally();
                    if (mine) reinterpret_cast<float4*>(P.data)[(long long)ly * P.pitch + lx] = make_float4(acc.C[0], acc.C[1], acc.C[2], acc.A);
                }
            }
        }
    }
    if (A.counters) {
        if (GLOBAL) count(A.counters, kRays, c_nom ? 1 : 0);
        count(A.counters, kNominal, c_nom);
        count(A.counters, kTaken, c_taken);
        count(A.counters, kVisited, c_nom ? 1 : 0);
        count(A.counters, kSkipped, c_reached - c_taken);
        count(A.counters, kTerminated, c_stopped);
    }
}

// ---------------------------------------------------------------------------------------------- dispatch
// V = float: every marcher, both layouts.  V = __half (VR_OPT_VOXEL_TYPE 1): layout 1 only and plain loads only
// (a 2-byte voxel cannot travel alone through the 4-byte cp.async ring): the lockstep marcher keeps its gathers in
// registers and the occupancy marcher gathers synchronously.
template <typename V>
constexpr bool kHalf = !std::is_same<V, float>::value;

// the occupancy marcher serves sparse emission-absorption on the micro-block layout
static bool use_occ_kernel(const CubeDesc& c, const RenderArgs& a) {
    return a.variant == 3 && a.mode == VR_MODE_EA && a.skip >= 3 && c.layout == 1;
}

// the same kernel with the macro-cell runs walked first and the occupancy test in step over the warp: dense rays
static bool use_runs_kernel(const CubeDesc& c, const RenderArgs& a) {
    return a.variant == 4 && a.mode == VR_MODE_EA && a.skip >= 3 && c.layout == 1;
}

template <typename V, bool GLOBAL, bool REGS, typename... Args>
static void launch_ls(const CubeDesc& c, const RenderArgs& a, dim3 grid, cudaStream_t s, Args... args) {
    if (a.mode == VR_MODE_MIP) {
        if constexpr (!kHalf<V>) { if (c.layout == 0) { render_ls_kernel<VR_MODE_MIP, 0, GLOBAL, false, REGS, V><<<grid, kThreads, 0, s>>>(args...); return; } }
        render_ls_kernel<VR_MODE_MIP, 1, GLOBAL, false, REGS, V><<<grid, kThreads, 0, s>>>(args...);
    } else if (a.dense) {
        if constexpr (!kHalf<V>) { if (c.layout == 0) { render_ls_kernel<VR_MODE_EA, 0, GLOBAL, true, REGS, V><<<grid, kThreads, 0, s>>>(args...); return; } }
        render_ls_kernel<VR_MODE_EA, 1, GLOBAL, true, REGS, V><<<grid, kThreads, 0, s>>>(args...);
    } else {
        if constexpr (!kHalf<V>) { if (c.layout == 0) { render_ls_kernel<VR_MODE_EA, 0, GLOBAL, false, REGS, V><<<grid, kThreads, 0, s>>>(args...); return; } }
        render_ls_kernel<VR_MODE_EA, 1, GLOBAL, false, REGS, V><<<grid, kThreads, 0, s>>>(args...);
    }
}

template <typename V, bool GLOBAL, typename... Args>
static void launch_ls_ring(const CubeDesc& c, const RenderArgs& a, dim3 grid, cudaStream_t s, Args... args) {
    if constexpr (kHalf<V>) launch_ls<V, GLOBAL, true>(c, a, grid, s, args...);
    else {
        if (a.ring) launch_ls<V, GLOBAL, true>(c, a, grid, s, args...);
        else launch_ls<V, GLOBAL, false>(c, a, grid, s, args...);
    }
}

template <typename V>
static cudaError_t launch_render_global_t(const CubeDesc& c, const ViewDesc& v, const TFDesc& t, const RenderArgs& a, cudaStream_t s) {
    dim3 grid((v.W + kTileW - 1) / kTileW, (v.H + kTileH - 1) / kTileH);
    const PartialDev* none = nullptr;
    if (use_occ_kernel(c, a)) { render_occ_kernel<true, V, !kHalf<V>><<<grid, kThreads, 0, s>>>(c, v, t, a, none, 0); return cudaGetLastError(); }
    if (use_runs_kernel(c, a)) { render_occ_kernel<true, V, !kHalf<V>, 1><<<grid, kThreads, 0, s>>>(c, v, t, a, none, 0); return cudaGetLastError(); }
    if (a.variant == 3) launch_ls_ring<V, true>(c, a, grid, s, c, v, t, a, none, 0);
    else if (a.mode == VR_MODE_EA && c.layout == 1 && a.skip >= 3 && v.step < kJumpStep)     // small steps: jump out of idle micro-blocks
        render_global_kernel<VR_MODE_EA, 1, true, V><<<grid, kThreads, 0, s>>>(c, v, t, a);
    else if (a.mode == VR_MODE_MIP) {
        if constexpr (!kHalf<V>) { if (c.layout == 0) { render_global_kernel<VR_MODE_MIP, 0, false, V><<<grid, kThreads, 0, s>>>(c, v, t, a); return cudaGetLastError(); } }
        render_global_kernel<VR_MODE_MIP, 1, false, V><<<grid, kThreads, 0, s>>>(c, v, t, a);
    } else {
        if constexpr (!kHalf<V>) { if (c.layout == 0) { render_global_kernel<VR_MODE_EA, 0, false, V><<<grid, kThreads, 0, s>>>(c, v, t, a); return cudaGetLastError(); } }
        render_global_kernel<VR_MODE_EA, 1, false, V><<<grid, kThreads, 0, s>>>(c, v, t, a);
    }
    return cudaGetLastError();
}

template <typename V>
static cudaError_t launch_render_bricks_t(const CubeDesc& c, const ViewDesc& v, const TFDesc& t, const RenderArgs& a,
                                          const PartialDev* d_partials, int n, int total_tiles, cudaStream_t s) {
    if (n == 0 || total_tiles == 0) return cudaSuccess;
    dim3 grid((v.W + kTileW - 1) / kTileW, (v.H + kTileH - 1) / kTileH);
    if (use_occ_kernel(c, a)) {
        render_occ_kernel<false, V, !kHalf<V>><<<grid, kThreads, 0, s>>>(c, v, t, a, d_partials, n);
        return cudaGetLastError();
    }
    if (use_runs_kernel(c, a)) {
        render_occ_kernel<false, V, !kHalf<V>, VR_DENSE_TEST><<<grid, kThreads, 0, s>>>(c, v, t, a, d_partials, n);
        return cudaGetLastError();
    }
    if (a.variant == 3) launch_ls_ring<V, false>(c, a, dim3(total_tiles), s, c, v, t, a, d_partials, n);
    else if (a.variant == 1) {
        if (a.mode == VR_MODE_MIP) {
            if constexpr (!kHalf<V>) { if (c.layout == 0) { render_bricks_kernel<VR_MODE_MIP, 0, V><<<total_tiles, kThreads, 0, s>>>(c, v, t, a, d_partials, n); return cudaGetLastError(); } }
            render_bricks_kernel<VR_MODE_MIP, 1, V><<<total_tiles, kThreads, 0, s>>>(c, v, t, a, d_partials, n);
        } else {
            if constexpr (!kHalf<V>) { if (c.layout == 0) { render_bricks_kernel<VR_MODE_EA, 0, V><<<total_tiles, kThreads, 0, s>>>(c, v, t, a, d_partials, n); return cudaGetLastError(); } }
            render_bricks_kernel<VR_MODE_EA, 1, V><<<total_tiles, kThreads, 0, s>>>(c, v, t, a, d_partials, n);
        }
    } else {
        if (a.mode == VR_MODE_EA && c.layout == 1 && a.skip >= 3 && v.step < kJumpStep)      // small steps: jump out of idle micro-blocks
            render_tiles_kernel<VR_MODE_EA, 1, true, V><<<grid, kThreads, 0, s>>>(c, v, t, a, d_partials, n);
        else if (a.mode == VR_MODE_MIP) {
            if constexpr (!kHalf<V>) { if (c.layout == 0) { render_tiles_kernel<VR_MODE_MIP, 0, false, V><<<grid, kThreads, 0, s>>>(c, v, t, a, d_partials, n); return cudaGetLastError(); } }
            render_tiles_kernel<VR_MODE_MIP, 1, false, V><<<grid, kThreads, 0, s>>>(c, v, t, a, d_partials, n);
        } else {
            if constexpr (!kHalf<V>) { if (c.layout == 0) { render_tiles_kernel<VR_MODE_EA, 0, false, V><<<grid, kThreads, 0, s>>>(c, v, t, a, d_partials, n); return cudaGetLastError(); } }
            render_tiles_kernel<VR_MODE_EA, 1, false, V><<<grid, kThreads, 0, s>>>(c, v, t, a, d_partials, n);
        }
    }
    return cudaGetLastError();
}

}  // namespace
}  // namespace vr
