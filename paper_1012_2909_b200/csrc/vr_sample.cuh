// Device-side building blocks of the ray marchers, shared by the kernels of vr_march.cu and
// vr_touch.cu (not part of the C ABI): O-2 ray set-up, O-3 lattice positions and brick membership, O-4
// trilinear gather, O-6 table lookup, O-7 front-to-back fold, run lengths and the O-10 activity tests.
//
// Arithmetic contract (readings O-2...O-7, O-11): the
// ray is set up in fp64 and rounded once to float32; every per-sample operation is an explicit
// IEEE float32 + - * fma floor min max compare (no fast-math, built with --fmad=false).
#pragma once
#include <cuda_fp16.h>

#include "vr_internal.cuh"

namespace vr {
namespace {


struct Ray {
    float o[3], d[3];
    float step;
    float margin;      // bound on |float32 position - exact position| (x8), voxels
    float inv[3];      // 1 / (step |d_a|)
    int k0, k1;        // exact interval of taken lattice indices (empty if k0 > k1)
};

__device__ __forceinline__ void unproject(const double* Mi, double xn, double yn, double zn, double out[3]) {
    double X = fma(Mi[0], xn, fma(Mi[1], yn, fma(Mi[2], zn, Mi[3])));
    double Y = fma(Mi[4], xn, fma(Mi[5], yn, fma(Mi[6], zn, Mi[7])));
    double Z = fma(Mi[8], xn, fma(Mi[9], yn, fma(Mi[10], zn, Mi[11])));
    double Wc = fma(Mi[12], xn, fma(Mi[13], yn, fma(Mi[14], zn, Mi[15])));
    out[0] = X / Wc; out[1] = Y / Wc; out[2] = Z / Wc;
}

__device__ __forceinline__ void position(const Ray& r, float kf, float p[3]) {
    float t = __fmul_rn(kf, r.step);                       // O-3: t_k = k * Delta
    p[0] = __fmaf_rn(t, r.d[0], r.o[0]);
    p[1] = __fmaf_rn(t, r.d[1], r.o[1]);
    p[2] = __fmaf_rn(t, r.d[2], r.o[2]);
}

__device__ __forceinline__ bool inside(const float p[3], const float hi[3]) {      // O-3 "taken"
    return p[0] >= 0.f && p[0] <= hi[0] && p[1] >= 0.f && p[1] <= hi[1] && p[2] >= 0.f && p[2] <= hi[2];
}

// O-2 ray of view pixel (i, j) and the exact interval [k0, k1] of its taken samples (O-3).
__device__ void setup_ray(const ViewDesc& V, const CubeDesc& c, int i, int j, Ray& r) {
    double xn = (2.0 * ((double)i + 0.5)) / (double)V.W - 1.0;
    double yn = 1.0 - (2.0 * ((double)j + 0.5)) / (double)V.H;
    double Pn[3], Pf[3];
    unproject(V.Minv, xn, yn, -1.0, Pn);
    unproject(V.Minv, xn, yn, +1.0, Pf);
    double dx = Pf[0] - Pn[0], dy = Pf[1] - Pn[1], dz = Pf[2] - Pn[2];
    double L = sqrt(fma(dx, dx, fma(dy, dy, dz * dz)));
    double d64[3] = {dx / L, dy / L, dz / L};
    r.step = V.step;
    float Lf = (float)L;
    double omax = 0.0;
    for (int a = 0; a < 3; ++a) {
        r.o[a] = (float)Pn[a]; r.d[a] = (float)d64[a];
        r.inv[a] = r.d[a] == 0.f ? 0.f : __frcp_rn(__fmul_rn(r.step, fabsf(r.d[a])));
        omax = fmax(omax, fabs(Pn[a]));
    }
    r.margin = (float)((omax + L) * (1.0 / 1048576.0));
    r.k0 = 0; r.k1 = -1;
    if (!(L > 0.0) || !isfinite(L)) return;
    // largest lattice index with t_k <= L (float32 compare, as the oracle)
    double q = floor((double)Lf / (double)r.step) + 2.0;
    if (!(q < 16000000.0)) return;                          // guard: absurd step / far plane
    int kmax = (int)q;
    while (kmax >= 0 && !(__fmul_rn((float)kmax, r.step) <= Lf)) --kmax;
    if (kmax < 0) return;
    // conservative bracket (fp64 slabs widened by the float32 error bound), then exact shrink with
    // the float32 predicate: positions are monotone in k per axis, so the taken set is an interval
    double t0 = 0.0, t1 = (double)kmax * (double)r.step;
    for (int a = 0; a < 3; ++a) {
        double eps = (fabs(Pn[a]) + L) * (1.0 / 1048576.0);
        if (fabs(d64[a]) < 1e-9) continue;
        double ta = (-eps - Pn[a]) / d64[a], tb = ((double)(c.N[a] - 1) + eps - Pn[a]) / d64[a];
        t0 = fmax(t0, fmin(ta, tb)); t1 = fmin(t1, fmax(ta, tb));
    }
    if (!(t0 <= t1 + 8.0 * (double)r.step)) return;
    int klo = max(0, (int)floor(t0 / (double)r.step) - 3);
    int khi = min(kmax, (int)ceil(t1 / (double)r.step) + 3);
    const float hi[3] = {(float)(c.N[0] - 1), (float)(c.N[1] - 1), (float)(c.N[2] - 1)};
    float p[3];
    while (klo <= khi) { position(r, (float)klo, p); if (inside(p, hi)) break; ++klo; }
    while (khi >= klo) { position(r, (float)khi, p); if (inside(p, hi)) break; --khi; }
    r.k0 = klo; r.k1 = khi;
}

// floor of 0 <= p < 2^23 without a conversion instruction: p + 2^23 rounded down is exact.
__device__ __forceinline__ int floor_pos(float p, float& fl) {
    float x = __fadd_rd(p, 8388608.0f);
    fl = __fsub_rn(x, 8388608.0f);
    return __float_as_int(x) - 0x4B000000;
}

__device__ __forceinline__ float lerp(float a, float b, float w) { return __fmaf_rn(w, __fsub_rn(b, a), a); }   // O-4

// One brick as the sampler sees it.  s0 / s1: layout 0 - row pitch P0 and plane pitch P0 P1;
// layout 1 - elements per row of micro-blocks (32 T0) and per plane of micro-blocks (32 T0 T1).
// V: the stored voxel type, float or __half (CubeDesc::vtype; VR_OPT_VOXEL_TYPE).  A __half voxel is converted to
// float32 when it is read (exact), everything after that is the same float32 arithmetic.
template <typename V>
struct BrickRefT {
    const V* base;
    int lo[3];
    unsigned s0, s1;
};
using BrickRef = BrickRefT<float>;

template <int LAYOUT, typename V = float>
__device__ __forceinline__ BrickRefT<V> brick_ref(const CubeDesc& c, int bid, const int lo[3]) {
    BrickRefT<V> b;
    b.base = reinterpret_cast<const V*>(c.cube) + (long long)bid * c.stride;
    b.lo[0] = lo[0]; b.lo[1] = lo[1]; b.lo[2] = lo[2];
    if (LAYOUT == 0) { b.s0 = (unsigned)c.P[0]; b.s1 = (unsigned)(c.P[0] * c.P[1]); }
    else { b.s0 = 32u * (unsigned)c.T[0]; b.s1 = 32u * (unsigned)(c.T[0] * c.T[1]); }
    return b;
}

__device__ __forceinline__ float load_voxel(const float* p) { return __ldg(p); }
__device__ __forceinline__ float load_voxel(const __half* p) { return __half2float(__ldg(p)); }

// Offset q of stored voxel (lx, ly, lz) inside its brick and the steps to its +1 neighbours.
template <int LAYOUT, typename V>
__device__ __forceinline__ void cell_address(const BrickRefT<V>& b, unsigned lx, unsigned ly, unsigned lz, unsigned& q,
                                             unsigned& dx, unsigned& dy, unsigned& dz) {
    if (LAYOUT == 0) {
        q = lx + b.s0 * ly + b.s1 * lz;
        dx = 1u; dy = b.s0; dz = b.s1;
    } else {                              // step to the +1 neighbour: inside the micro-block or into the next one
        q = ((lx >> 2) << 5) + (lx & 3u) + (ly >> 2) * b.s0 + ((ly & 2u) << 3) + ((ly & 1u) << 2) + (lz >> 1) * b.s1 + ((lz & 1u) << 3);
        dx = (lx & 3u) == 3u ? 29u : 1u;
        dy = (ly & 1u) == 0u ? 4u : ((ly & 2u) == 0u ? 12u : b.s0 - 20u);
        dz = (lz & 1u) ? b.s1 - 8u : 8u;
    }
}

// The 8 voxels of the trilinear cell whose lower corner is (ix, iy, iz) (global voxel indices,
// inside brick b or on its halo), in the order 000 100 010 110 001 101 011 111.
template <int LAYOUT, typename V>
__device__ __forceinline__ void gather8(const BrickRefT<V>& b, int ix, int iy, int iz, float v[8]) {
    const unsigned lx = (unsigned)(ix - b.lo[0]), ly = (unsigned)(iy - b.lo[1]), lz = (unsigned)(iz - b.lo[2]);
    unsigned q, dx, dy, dz;
    cell_address<LAYOUT>(b, lx, ly, lz, q, dx, dy, dz);
    const V* p = b.base + q;
    v[0] = load_voxel(p);           v[1] = load_voxel(p + dx);
    v[2] = load_voxel(p + dy);      v[3] = load_voxel(p + dy + dx);
    v[4] = load_voxel(p + dz);      v[5] = load_voxel(p + dz + dx);
    v[6] = load_voxel(p + dz + dy); v[7] = load_voxel(p + dz + dy + dx);
}

__device__ __forceinline__ float trilinear(const float v[8], float wx, float wy, float wz) {   // O-4: x, then y, then z
    const float c00 = lerp(v[0], v[1], wx), c10 = lerp(v[2], v[3], wx);
    const float c01 = lerp(v[4], v[5], wx), c11 = lerp(v[6], v[7], wx);
    return lerp(lerp(c00, c10, wy), lerp(c01, c11, wy), wz);
}

template <int LAYOUT, typename V>
__device__ __forceinline__ float sample(const BrickRefT<V>& b, const float p[3]) {
    float fx, fy, fz, v[8];
    const int ix = floor_pos(p[0], fx), iy = floor_pos(p[1], fy), iz = floor_pos(p[2], fz);
    gather8<LAYOUT>(b, ix, iy, iz, v);
    return trilinear(v, __fsub_rn(p[0], fx), __fsub_rn(p[1], fy), __fsub_rn(p[2], fz));
}

struct Accum { float C[3]; float A; float m; };

// O-6 lookup of table coordinate x (already scaled, not yet clamped) in the baked table.
__device__ __forceinline__ float4 tf_at(const float4* __restrict__ tab, float x) {
    x = fminf(fmaxf(x, 0.f), 255.f);
    float fl;
    const int i = min(floor_pos(x, fl), 254);
    const float f = __fsub_rn(x, fminf(fl, 254.f));
    const float4 a = tab[i], b = tab[i + 1];
    return make_float4(lerp(a.x, b.x, f), lerp(a.y, b.y, f), lerp(a.z, b.z, f), lerp(a.w, b.w, f));
}

__device__ __forceinline__ bool over(Accum& acc, float cr, float cg, float cb, float ca, float tau) {   // O-7
    const float w = __fmul_rn(__fsub_rn(1.f, acc.A), ca);
    acc.C[0] = __fmaf_rn(w, cr, acc.C[0]);
    acc.C[1] = __fmaf_rn(w, cg, acc.C[1]);
    acc.C[2] = __fmaf_rn(w, cb, acc.C[2]);
    acc.A = __fadd_rn(acc.A, w);
    return acc.A >= tau;
}

// O-5 / O-6 / O-7: fold one sample value into the ray's accumulator.  A sample whose table
// coordinate x lies below T.x_clear falls between two entries of zero opacity: its weight
// w = (1 - A) * 0 is exactly zero and leaves C and A unchanged, so the lookup is not done.
template <int MODE>
__device__ __forceinline__ bool fold(Accum& acc, float v, const float4* tab, const TFDesc& T, float tau) {
    if (MODE == VR_MODE_MIP) { acc.m = fmaxf(acc.m, v); return false; }
    const float x = __fmul_rn(__fsub_rn(v, T.vmin), T.scale);
    if (x < T.x_clear) return false;
    const float4 q = tf_at(tab, x);
    return over(acc, q.x, q.y, q.z, q.w, tau);
}

// Conservative number (>= 1) of samples, starting at the one at p, whose floor(position) stays in
// the aligned box [lo, lo + S).
__device__ __forceinline__ int run_length(const Ray& r, const float p[3], const int lo[3], const int S[3]) {
    float q = 1.0e9f;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        if (r.d[a] == 0.f) continue;
        float dist = r.d[a] > 0.f ? __fsub_rn((float)(lo[a] + S[a]), p[a]) : __fsub_rn(p[a], (float)lo[a]);
        q = fminf(q, __fmul_rn(fmaxf(__fsub_rn(dist, r.margin), 0.f), r.inv[a]));
    }
    return 1 + (int)(q * 0.9999f);
}

__device__ __forceinline__ void brick_of(const CubeDesc& c, const int i[3], int b[3]) {
#pragma unroll
    for (int a = 0; a < 3; ++a) b[a] = c.sh[a] >= 0 ? (i[a] >> c.sh[a]) : (i[a] / c.B[a]);
}

__device__ __forceinline__ void load_tf(float4* tab, const float4* src) {
    for (int i = threadIdx.x; i < 256; i += blockDim.x) tab[i] = src[i];
    __syncthreads();
}

__device__ __forceinline__ void count(unsigned long long* counters, int which, unsigned long long v) {
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    if ((threadIdx.x & 31) == 0 && v) atomicAdd(counters + which, v);
}

__device__ __forceinline__ void tile_pixel(int& tx, int& ty) {     // warp = 8 x 4 pixels
    int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    tx = (warp & 1) * 8 + (lane & 7);
    ty = (warp >> 1) * 4 + (lane >> 3);
}

// Shrink the taken interval [ka, kb] of ray r to its members of the box of cells [lo, lo + ext), i.e. the samples
// with lo_a <= floor(p_a) < lo_a + ext_a (O-3: for a brick, floor(p_a) / B_a == b_a): conservative float32
// bracket of the box's slab interval, then exact shrink with the membership predicate, which is monotone per axis.
__device__ __forceinline__ void box_interval(const Ray& r, const int lo[3], const int ext[3], int& ka, int& kb) {
    if (ka > kb) return;
    // in units of the lattice index: r.inv = 1 / (step |d|), no division
    float t0 = 0.f, t1 = 3.0e38f;
    bool empty = false;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        float flo = (float)lo[a] - r.margin, fhi = (float)(lo[a] + ext[a]) + r.margin;
        if (r.d[a] == 0.f) { if (r.o[a] < flo || r.o[a] > fhi) empty = true; continue; }
        const float si = r.d[a] > 0.f ? r.inv[a] : -r.inv[a];
        float ta = __fmul_rn(flo - r.o[a], si), tb = __fmul_rn(fhi - r.o[a], si);
        t0 = fmaxf(t0, fminf(ta, tb)); t1 = fminf(t1, fmaxf(ta, tb));
    }
    if (empty || !(t0 <= t1)) { ka = 0; kb = -1; return; }
    float qa = floorf(t0) - 2.f, qb = ceilf(t1) + 2.f;
    ka = max(ka, (int)fminf(fmaxf(qa, 0.f), 1.0e9f));
    kb = min(kb, (int)fminf(fmaxf(qb, -1.f), 1.0e9f));
    float p[3], fl;
    while (ka <= kb) {
        position(r, (float)ka, p);                          // floor(p_a) / B_a == b_a  <=>  lo_a <= floor(p_a) < lo_a + B_a
        if ((unsigned)(floor_pos(p[0], fl) - lo[0]) < (unsigned)ext[0] && (unsigned)(floor_pos(p[1], fl) - lo[1]) < (unsigned)ext[1] &&
            (unsigned)(floor_pos(p[2], fl) - lo[2]) < (unsigned)ext[2]) break;
        ++ka;
    }
    while (kb >= ka) {
        position(r, (float)kb, p);
        if ((unsigned)(floor_pos(p[0], fl) - lo[0]) < (unsigned)ext[0] && (unsigned)(floor_pos(p[1], fl) - lo[1]) < (unsigned)ext[1] &&
            (unsigned)(floor_pos(p[2], fl) - lo[2]) < (unsigned)ext[2]) break;
        --kb;
    }
}

__device__ __forceinline__ void brick_interval(const CubeDesc& c, const Ray& r, const int b[3], const int lo[3], int& ka, int& kb) {
    (void)b;
    box_interval(r, lo, c.B, ka, kb);
}

// Which partial does this CTA's tile belong to, and which pixel of it is this thread's.
__device__ __forceinline__ bool locate_tile(const PartialDev* __restrict__ parts, int n_parts, PartialDev& part, int& lx, int& ly) {
    if (threadIdx.x == 0) {
        int lo = 0, hi = n_parts - 1;
        const int tile = blockIdx.x;
        while (lo < hi) { int mid = (lo + hi + 1) >> 1; if (parts[mid].tile0 <= tile) lo = mid; else hi = mid - 1; }
        part = parts[lo];
    }
    __syncthreads();
    int tx, ty; tile_pixel(tx, ty);
    const int tiles_x = (part.w + kTileW - 1) / kTileW;
    const int tile = blockIdx.x - part.tile0;
    lx = (tile % tiles_x) * kTileW + tx; ly = (tile / tiles_x) * kTileH + ty;
    return lx < part.w && ly < part.h;
}

// O-10 at the 8^3 macro-cell level for the sample whose cell has lower corner (ix, iy, iz) in
// brick bid: true if the sample cannot contribute.  EA: every table entry the cell's value range
// can touch has zero opacity (one bit per cell, classify_cells_kernel); MIP: the cell's maximum
// cannot raise m.
template <int MODE>
__device__ __forceinline__ bool cell_idle(const CubeDesc& c, int bid, const int lo[3], int ix, int iy, int iz, float m) {
    const int cidx = ((ix - lo[0]) >> 3) + c.C[0] * (((iy - lo[1]) >> 3) + c.C[1] * ((iz - lo[2]) >> 3));
    if (MODE == VR_MODE_MIP) return __ldg(&c.cell_mm[(long long)bid * c.cells_per_brick + cidx]).y <= m;
    return ((__ldg(&c.cell_bits[(long long)bid * c.cell_words_per_brick + (cidx >> 5)]) >> (cidx & 31)) & 1u) == 0u;
}

// Occupancy word and bit (CubeDesc::occ) of the trilinear cell whose lower corner is stored voxel (lx, ly, lz) of a
// brick: the word of its micro-block (= the index of the block's line in the brick), the voxel's slot in the line.
__device__ __forceinline__ unsigned occ_word_index(const CubeDesc& c, unsigned lx, unsigned ly, unsigned lz) {
    return (lx >> 2) + (unsigned)c.T[0] * ((ly >> 2) + (unsigned)c.T[1] * (lz >> 1));
}
__device__ __forceinline__ unsigned occ_bit_index(unsigned lx, unsigned ly, unsigned lz) {
    return (lx & 3u) + ((ly & 1u) << 2) + ((lz & 1u) << 3) + ((ly & 2u) << 3);
}

constexpr float kJumpStep = 0.4f;
struct Stats { unsigned long long taken, visit, skip; };

}  // namespace
}  // namespace vr
