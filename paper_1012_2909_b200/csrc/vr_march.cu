// The ray marcher (BASELINE.json north_star (2)): per-pixel rays through the
// brick-major cube, fixed step, trilinear interpolation, MIP or front-to-back emission-absorption
// through the 256-entry transfer function with early ray termination, min/max brick skipping.
//
// Arithmetic contract (readings O-2...O-7, O-11): the
// ray is set up in fp64 and rounded once to float32; every per-sample operation is an explicit
// IEEE float32 + - * fma floor min max compare (no fast-math, built with --fmad=false), so frames
// agree with the float32 instantiation of the oracle to the bit and with its fp64 instantiation
// within BASELINE.json's tolerances.
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

// The 8 corner voxels of the trilinear cell a ray is in, kept in registers between samples
// (DESIGN.md "Cell cache").  With a step of half a voxel consecutive samples mostly fall in the
// same cell or in a face neighbour, so a sample needs 0 or 4 new voxels instead of 8.  The values
// are the voxels themselves, so the interpolated result does not depend on the cache.
struct Cell {
    float c000, c100, c010, c110, c001, c101, c011, c111;
    int ix, iy, iz;                       // cell index (global voxel coordinates); ix < 0: invalid
};
constexpr int kNoCell = -(1 << 30);

struct BrickRef {
    const float* base;     // first float of the brick
    unsigned off0;         // lo0 + P0 lo1 + P01 lo2 (mod 2^32): subtracting it makes offsets brick-local
    unsigned P0, P01;
};

__device__ __forceinline__ unsigned voxel_offset(const BrickRef& b, int ix, int iy, int iz) {
    return (unsigned)ix + b.P0 * (unsigned)iy + b.P01 * (unsigned)iz - b.off0;
}

__device__ __forceinline__ void cell_load_all(const BrickRef& b, int ix, int iy, int iz, Cell& cc) {
    const float* q = b.base + voxel_offset(b, ix, iy, iz);
    cc.c000 = __ldg(q);                 cc.c100 = __ldg(q + 1);
    cc.c010 = __ldg(q + b.P0);          cc.c110 = __ldg(q + b.P0 + 1);
    cc.c001 = __ldg(q + b.P01);         cc.c101 = __ldg(q + b.P01 + 1);
    cc.c011 = __ldg(q + b.P01 + b.P0);  cc.c111 = __ldg(q + b.P01 + b.P0 + 1);
}

// Move the cached cell to (ix, iy, iz): one face shift (4 new voxels) per axis that moved by one,
// through the intermediate cells (ix, cy, cz) -> (ix, iy, cz) -> (ix, iy, iz), all of which lie in
// the brick because the old and the new cell do.  Anything else reloads the 8 voxels.
__device__ __forceinline__ void cell_move(const BrickRef& b, int ix, int iy, int iz, Cell& cc) {
    const int ddx = ix - cc.ix, ddy = iy - cc.iy, ddz = iz - cc.iz;
    if ((unsigned)(ddx + 1) <= 2u && (unsigned)(ddy + 1) <= 2u && (unsigned)(ddz + 1) <= 2u) {
        if (ddx != 0) {
            const float* q = b.base + voxel_offset(b, ix, cc.iy, cc.iz);
            if (ddx > 0) {
                cc.c000 = cc.c100; cc.c010 = cc.c110; cc.c001 = cc.c101; cc.c011 = cc.c111;
                cc.c100 = __ldg(q + 1);         cc.c110 = __ldg(q + b.P0 + 1);
                cc.c101 = __ldg(q + b.P01 + 1); cc.c111 = __ldg(q + b.P01 + b.P0 + 1);
            } else {
                cc.c100 = cc.c000; cc.c110 = cc.c010; cc.c101 = cc.c001; cc.c111 = cc.c011;
                cc.c000 = __ldg(q);             cc.c010 = __ldg(q + b.P0);
                cc.c001 = __ldg(q + b.P01);     cc.c011 = __ldg(q + b.P01 + b.P0);
            }
        }
        if (ddy != 0) {
            const float* q = b.base + voxel_offset(b, ix, iy, cc.iz);
            if (ddy > 0) {
                cc.c000 = cc.c010; cc.c100 = cc.c110; cc.c001 = cc.c011; cc.c101 = cc.c111;
                cc.c010 = __ldg(q + b.P0);          cc.c110 = __ldg(q + b.P0 + 1);
                cc.c011 = __ldg(q + b.P01 + b.P0);  cc.c111 = __ldg(q + b.P01 + b.P0 + 1);
            } else {
                cc.c010 = cc.c000; cc.c110 = cc.c100; cc.c011 = cc.c001; cc.c111 = cc.c101;
                cc.c000 = __ldg(q);                 cc.c100 = __ldg(q + 1);
                cc.c001 = __ldg(q + b.P01);         cc.c101 = __ldg(q + b.P01 + 1);
            }
        }
        if (ddz != 0) {
            const float* q = b.base + voxel_offset(b, ix, iy, iz);
            if (ddz > 0) {
                cc.c000 = cc.c001; cc.c100 = cc.c101; cc.c010 = cc.c011; cc.c110 = cc.c111;
                cc.c001 = __ldg(q + b.P01);         cc.c101 = __ldg(q + b.P01 + 1);
                cc.c011 = __ldg(q + b.P01 + b.P0);  cc.c111 = __ldg(q + b.P01 + b.P0 + 1);
            } else {
                cc.c001 = cc.c000; cc.c101 = cc.c100; cc.c011 = cc.c010; cc.c111 = cc.c110;
                cc.c000 = __ldg(q);                 cc.c100 = __ldg(q + 1);
                cc.c010 = __ldg(q + b.P0);          cc.c110 = __ldg(q + b.P0 + 1);
            }
        }
    } else {
        cell_load_all(b, ix, iy, iz, cc);
    }
    cc.ix = ix; cc.iy = iy; cc.iz = iz;
}

// O-4 trilinear at p (floor(p) inside brick b).  VAR 0 reads the 8 voxels of every sample, VAR 1
// goes through the cell cache.
template <int VAR>
__device__ __forceinline__ float sample(const BrickRef& b, const float p[3], Cell& cc) {
    float fx, fy, fz;
    const int ix = floor_pos(p[0], fx), iy = floor_pos(p[1], fy), iz = floor_pos(p[2], fz);
    const float wx = __fsub_rn(p[0], fx), wy = __fsub_rn(p[1], fy), wz = __fsub_rn(p[2], fz);
    if (VAR == 0) cell_load_all(b, ix, iy, iz, cc);
    else if (ix != cc.ix || iy != cc.iy || iz != cc.iz) cell_move(b, ix, iy, iz, cc);
    const float c00 = lerp(cc.c000, cc.c100, wx), c10 = lerp(cc.c010, cc.c110, wx);
    const float c01 = lerp(cc.c001, cc.c101, wx), c11 = lerp(cc.c011, cc.c111, wx);
    const float c0 = lerp(c00, c10, wy), c1 = lerp(c01, c11, wy);
    return lerp(c0, c1, wz);
}

struct Accum { float C[3]; float A; float m; };

// O-5 / O-6 / O-7: fold one sample value into the ray's accumulator.  A sample whose table
// coordinate x lies below T.x_clear falls between two entries of zero opacity: its weight
// w = (1 - A) * 0 is exactly zero and leaves C and A unchanged, so the lookup is not done.
template <int MODE>
__device__ __forceinline__ bool fold(Accum& acc, float v, const float4* tab, const TFDesc& T, float tau) {
    if (MODE == VR_MODE_MIP) { acc.m = fmaxf(acc.m, v); return false; }
    float x = __fmul_rn(__fsub_rn(v, T.vmin), T.scale);
    if (x < T.x_clear) return false;
    x = fminf(fmaxf(x, 0.f), 255.f);
    float fl;
    const int i = min(floor_pos(x, fl), 254);
    const float f = __fsub_rn(x, fminf(fl, 254.f));
    const float4 a = tab[i], b = tab[i + 1];
    const float qa = lerp(a.w, b.w, f);
    const float w = __fmul_rn(__fsub_rn(1.f, acc.A), qa);        // O-7
    acc.C[0] = __fmaf_rn(w, lerp(a.x, b.x, f), acc.C[0]);
    acc.C[1] = __fmaf_rn(w, lerp(a.y, b.y, f), acc.C[1]);
    acc.C[2] = __fmaf_rn(w, lerp(a.z, b.z, f), acc.C[2]);
    acc.A = __fadd_rn(acc.A, w);
    return acc.A >= tau;
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

// Shrink the taken interval [ka, kb] of ray r to its members of brick b (O-3): conservative float32
// bracket of the brick's slab interval, then exact shrink with the membership predicate
// floor(p_a) / B_a == b_a, which is monotone per axis.
__device__ __forceinline__ void brick_interval(const CubeDesc& c, const Ray& r, const int b[3], const int lo[3], int& ka, int& kb) {
    if (ka > kb) return;
    float t0 = 0.f, t1 = 3.0e38f;
    bool empty = false;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        float flo = (float)lo[a] - r.margin, fhi = (float)(lo[a] + c.B[a]) + r.margin;
        if (r.d[a] == 0.f) { if (r.o[a] < flo || r.o[a] > fhi) empty = true; continue; }
        float ta = (flo - r.o[a]) / r.d[a], tb = (fhi - r.o[a]) / r.d[a];
        t0 = fmaxf(t0, fminf(ta, tb)); t1 = fminf(t1, fmaxf(ta, tb));
    }
    if (empty || !(t0 <= t1)) { ka = 0; kb = -1; return; }
    float qa = floorf(t0 / r.step) - 2.f, qb = ceilf(t1 / r.step) + 2.f;
    ka = max(ka, (int)fminf(fmaxf(qa, 0.f), 1.0e9f));
    kb = min(kb, (int)fminf(fmaxf(qb, -1.f), 1.0e9f));
    float p[3], fl;
    while (ka <= kb) {
        position(r, (float)ka, p);
        int iv[3] = {floor_pos(p[0], fl), floor_pos(p[1], fl), floor_pos(p[2], fl)};
        int bb[3]; brick_of(c, iv, bb);
        if (bb[0] == b[0] && bb[1] == b[1] && bb[2] == b[2]) break;
        ++ka;
    }
    while (kb >= ka) {
        position(r, (float)kb, p);
        int iv[3] = {floor_pos(p[0], fl), floor_pos(p[1], fl), floor_pos(p[2], fl)};
        int bb[3]; brick_of(c, iv, bb);
        if (bb[0] == b[0] && bb[1] == b[1] && bb[2] == b[2]) break;
        --kb;
    }
}

struct Stats { unsigned long long taken, visit, skip; };

__device__ __forceinline__ BrickRef brick_ref(const CubeDesc& c, int bid, const int lo[3]) {
    BrickRef b;
    b.base = c.cube + (long long)bid * c.stride;
    b.P0 = (unsigned)c.P[0]; b.P01 = (unsigned)(c.P[0] * c.P[1]);
    b.off0 = (unsigned)lo[0] + b.P0 * (unsigned)lo[1] + b.P01 * (unsigned)lo[2];
    return b;
}

// March the lattice samples k .. ke (all of them members of brick `bid`, O-3) into `acc`.  With
// A.skip >= 2 the interval is cut into runs inside 8^3 macro-cells and a run is skipped when its
// cell cannot contribute (O-10, exact): EA - every table entry its value range can touch has zero
// opacity (bit precomputed per transfer function); MIP - the cell's maximum cannot raise m.
// Returns true if early ray termination fired.
template <int MODE, int VAR>
__device__ __forceinline__ bool march_interval(const CubeDesc& c, const Ray& r, const TFDesc& T, const RenderArgs& A,
                                               const float4* tab, int bid, const int lo[3], int k, int ke,
                                               Accum& acc, Stats& st) {
    const BrickRef b = brick_ref(c, bid, lo);
    const int S8[3] = {kCell, kCell, kCell};
    Cell cc;
    cc.ix = cc.iy = cc.iz = kNoCell;
    float kf = (float)k;                                    // exact: k < 2^24
    while (k <= ke) {
        int n = ke - k + 1;
        if (A.skip >= 2) {
            float p[3], fl;
            position(r, kf, p);
            const int cl[3] = {(floor_pos(p[0], fl) - lo[0]) >> 3, (floor_pos(p[1], fl) - lo[1]) >> 3,
                               (floor_pos(p[2], fl) - lo[2]) >> 3};
            const int clo[3] = {lo[0] + (cl[0] << 3), lo[1] + (cl[1] << 3), lo[2] + (cl[2] << 3)};
            n = min(n, run_length(r, p, clo, S8));
            const int cidx = cl[0] + c.C[0] * (cl[1] + c.C[1] * cl[2]);
            bool skip;
            if (MODE == VR_MODE_MIP) skip = __ldg(&c.cell_mm[(long long)bid * c.cells_per_brick + cidx]).y <= acc.m;
            else skip = ((__ldg(&c.cell_bits[(long long)bid * c.cell_words_per_brick + (cidx >> 5)]) >> (cidx & 31)) & 1u) == 0u;
            if (skip) { k += n; kf = __fadd_rn(kf, (float)n); ++st.skip; continue; }
        }
        ++st.visit;
        for (const int e = k + n; k < e; ++k, kf = __fadd_rn(kf, 1.f)) {
            float p[3];
            position(r, kf, p);
            const float v = sample<VAR>(b, p, cc);
            ++st.taken;
            if (fold<MODE>(acc, v, tab, T, A.tau)) return true;
        }
    }
    return false;
}

// ---------------------------------------------------------------- whole frame, O-8 GLOBAL
template <int MODE, int VAR>
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
        if (march_interval<MODE, VAR>(c, r, T, A, tab, bid, lo, k, k + n - 1, acc, st)) { stopped = true; break; }
        k += n;
    }
    if (live) {
        const long long px = (long long)(V.vy0 + j) * V.pitch + (V.vx0 + i);
        if (MODE == VR_MODE_MIP) {
            const bool any = r.k1 >= r.k0;
            A.out[px] = any ? acc.m : A.miss;
            if (A.out_rgba) {
                float4 q = make_float4(0.f, 0.f, 0.f, 0.f);
                if (any) {
                    float x = __fmul_rn(__fsub_rn(acc.m, T.vmin), T.scale);
                    x = fminf(fmaxf(x, 0.f), 255.f);
                    float fl; int ii = min(floor_pos(x, fl), 254);
                    float f = __fsub_rn(x, (float)ii);
                    float4 a = T.raw[ii], bb = T.raw[ii + 1];
                    q = make_float4(lerp(a.x, bb.x, f), lerp(a.y, bb.y, f), lerp(a.z, bb.z, f), lerp(a.w, bb.w, f));
                }
                reinterpret_cast<float4*>(A.out_rgba)[px] = q;
            }
        } else {                                           // O-7: premultiplied colour over bg
            float t = __fsub_rn(1.f, acc.A);
            float4 o = make_float4(__fmaf_rn(t, A.bg[0], acc.C[0]), __fmaf_rn(t, A.bg[1], acc.C[1]),
                                   __fmaf_rn(t, A.bg[2], acc.C[2]), __fmaf_rn(t, A.bg[3], acc.A));
            reinterpret_cast<float4*>(A.out)[px] = o;
        }
    }
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
template <int MODE, int VAR>
__global__ void __launch_bounds__(kThreads)
render_bricks_kernel(const __grid_constant__ CubeDesc c, const __grid_constant__ ViewDesc V,
                     const __grid_constant__ TFDesc T, const __grid_constant__ RenderArgs A,
                     const PartialDev* __restrict__ parts, int n_parts) {
    __shared__ float4 tab[256];
    __shared__ PartialDev part;
    if (threadIdx.x == 0) {           // which partial does this CTA's tile belong to?
        int lo = 0, hi = n_parts - 1;
        const int tile = blockIdx.x;
        while (lo < hi) { int mid = (lo + hi + 1) >> 1; if (parts[mid].tile0 <= tile) lo = mid; else hi = mid - 1; }
        part = parts[lo];
    }
    if (MODE == VR_MODE_EA) load_tf(tab, T.baked); else __syncthreads();
    int tx, ty; tile_pixel(tx, ty);
    const int tiles_x = (part.w + kTileW - 1) / kTileW;
    const int tile = blockIdx.x - part.tile0;
    const int lx = (tile % tiles_x) * kTileW + tx, ly = (tile / tiles_x) * kTileH + ty;
    const bool live = lx < part.w && ly < part.h;
    Ray r; r.k0 = 0; r.k1 = -1;
    if (live) setup_ray(V, c, part.x0 + lx, part.y0 + ly, r);
    const int bid = part.brick;
    const int b[3] = {bid % c.G[0], (bid / c.G[0]) % c.G[1], bid / (c.G[0] * c.G[1])};
    const int lo[3] = {b[0] * c.B[0], b[1] * c.B[1], b[2] * c.B[2]};
    int ka = r.k0, kb = r.k1;
    brick_interval(c, r, b, lo, ka, kb);
    Accum acc = {{0.f, 0.f, 0.f}, 0.f, -INFINITY};
    Stats st = {0, 0, 0};
    const bool stopped = march_interval<MODE, VAR>(c, r, T, A, tab, bid, lo, ka, kb, acc, st);
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

// ---------------------------------------------------------------- sort-last, one ray per warp
// Variant 2 ("sample-parallel").  The 128 threads of a CTA first set up
// the 128 rays of their pixel tile exactly as above (one ray per thread).  Then every warp walks
// through its own 32 rays one after the other, and the 32 lanes take 32 CONSECUTIVE lattice
// samples k .. k+31 of that one ray: positions, voxel gathers and trilinear interpolation run in
// parallel, and the lanes' addresses follow the ray, so every 32-byte sector the ray needs is
// fetched once and used at once - nothing has to survive in L1/L2 between iterations, whatever
// the view direction.  The front-to-back fold stays sequential in k (O-7): opaque samples are
// picked out with a ballot and folded in ascending order through shuffles, all lanes keeping the
// same accumulator; transparent samples (x < x_clear) contribute exact zeros and are not folded.
// MIP folds with a warp maximum (exact in any order).
template <int MODE>
__global__ void __launch_bounds__(kThreads)
render_bricks_sp_kernel(const __grid_constant__ CubeDesc c, const __grid_constant__ ViewDesc V,
                        const __grid_constant__ TFDesc T, const __grid_constant__ RenderArgs A,
                        const PartialDev* __restrict__ parts, int n_parts) {
    __shared__ float4 tab[256];
    __shared__ PartialDev part;
    if (threadIdx.x == 0) {
        int lo = 0, hi = n_parts - 1;
        const int tile = blockIdx.x;
        while (lo < hi) { int mid = (lo + hi + 1) >> 1; if (parts[mid].tile0 <= tile) lo = mid; else hi = mid - 1; }
        part = parts[lo];
    }
    if (MODE == VR_MODE_EA) load_tf(tab, T.baked); else __syncthreads();
    int tx, ty; tile_pixel(tx, ty);
    const int tiles_x = (part.w + kTileW - 1) / kTileW;
    const int tile = blockIdx.x - part.tile0;
    const int lx = (tile % tiles_x) * kTileW + tx, ly = (tile / tiles_x) * kTileH + ty;
    const bool live = lx < part.w && ly < part.h;
    Ray r; r.k0 = 0; r.k1 = -1;
    r.o[0] = r.o[1] = r.o[2] = 0.f; r.d[0] = r.d[1] = r.d[2] = 0.f; r.step = V.step; r.margin = 0.f;
    if (live) setup_ray(V, c, part.x0 + lx, part.y0 + ly, r);
    const int bid = part.brick;
    const int b[3] = {bid % c.G[0], (bid / c.G[0]) % c.G[1], bid / (c.G[0] * c.G[1])};
    const int lo[3] = {b[0] * c.B[0], b[1] * c.B[1], b[2] * c.B[2]};
    int ka = r.k0, kb = r.k1;
    brick_interval(c, r, b, lo, ka, kb);
    const BrickRef br = brick_ref(c, bid, lo);
    const int lane = threadIdx.x & 31;
    Accum mine = {{0.f, 0.f, 0.f}, 0.f, -INFINITY};
    unsigned long long n_taken = 0, n_term = 0, n_visit = 0;
    const unsigned todo = __ballot_sync(0xffffffffu, ka <= kb);
    for (unsigned rays = todo; rays; rays &= rays - 1) {
        const int src = __ffs(rays) - 1;
        Ray q;
        q.step = r.step;
#pragma unroll
        for (int a = 0; a < 3; ++a) { q.o[a] = __shfl_sync(0xffffffffu, r.o[a], src); q.d[a] = __shfl_sync(0xffffffffu, r.d[a], src); }
        const int qa = __shfl_sync(0xffffffffu, ka, src), qb = __shfl_sync(0xffffffffu, kb, src);
        Accum acc = {{0.f, 0.f, 0.f}, 0.f, -INFINITY};
        bool stopped = false;
        for (int k0 = qa; k0 <= qb && !stopped; k0 += 32) {
            const int k = k0 + lane;
            const bool act = k <= qb;
            float p[3];
            position(q, (float)min(k, qb), p);               // idle lanes repeat the last sample
            Cell cc;
            const float v = sample<0>(br, p, cc);
            if (MODE == VR_MODE_MIP) {
                float m = act ? v : -INFINITY;
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, o));
                acc.m = fmaxf(acc.m, m);
                if (lane == 0) n_taken += (unsigned long long)(min(qb - k0, 31) + 1);
            } else {
                float x = __fmul_rn(__fsub_rn(v, T.vmin), T.scale);
                const bool opaque = act && !(x < T.x_clear);
                unsigned bits = __ballot_sync(0xffffffffu, opaque);
                int n_here = min(qb - k0, 31) + 1;
                if (bits) {
                    float4 col = make_float4(0.f, 0.f, 0.f, 0.f);
                    if (opaque) {                           // O-6 lookup, one sample per lane
                        x = fminf(fmaxf(x, 0.f), 255.f);
                        float fl;
                        const int i = min(floor_pos(x, fl), 254);
                        const float f = __fsub_rn(x, fminf(fl, 254.f));
                        const float4 ta = tab[i], tb = tab[i + 1];
                        col = make_float4(lerp(ta.x, tb.x, f), lerp(ta.y, tb.y, f), lerp(ta.z, tb.z, f), lerp(ta.w, tb.w, f));
                    }
                    while (bits) {                          // O-7, ascending k
                        const int j = __ffs(bits) - 1;
                        bits &= bits - 1;
                        const float cr = __shfl_sync(0xffffffffu, col.x, j), cg = __shfl_sync(0xffffffffu, col.y, j);
                        const float cb = __shfl_sync(0xffffffffu, col.z, j), ca = __shfl_sync(0xffffffffu, col.w, j);
                        const float w = __fmul_rn(__fsub_rn(1.f, acc.A), ca);
                        acc.C[0] = __fmaf_rn(w, cr, acc.C[0]);
                        acc.C[1] = __fmaf_rn(w, cg, acc.C[1]);
                        acc.C[2] = __fmaf_rn(w, cb, acc.C[2]);
                        acc.A = __fadd_rn(acc.A, w);
                        if (acc.A >= A.tau) { stopped = true; n_here = j + 1; break; }
                    }
                }
                if (lane == 0) n_taken += (unsigned long long)n_here;
            }
        }
        if (lane == 0) { ++n_visit; n_term += stopped ? 1 : 0; }
        if (lane == src) mine = acc;
    }
    if (live) {
        const long long px = (long long)ly * part.pitch + lx;
        if (MODE == VR_MODE_MIP) reinterpret_cast<float*>(part.data)[px] = mine.m;
        else reinterpret_cast<float4*>(part.data)[px] = make_float4(mine.C[0], mine.C[1], mine.C[2], mine.A);
    }
    if (A.counters) {
        count(A.counters, kNominal, kb >= ka ? (unsigned long long)(kb - ka + 1) : 0ULL);
        count(A.counters, kTaken, n_taken);
        count(A.counters, kVisited, n_visit);
        count(A.counters, kTerminated, n_term);
    }
}

// O-10 per transfer function: one bit per 8^3 macro-cell, set iff a table entry that the cell's
// value range [min, max] (halo-inclusive) can touch has non-zero opacity.  `nz` is the running
// count of entries with non-zero baked opacity, so the range test is one subtraction.
struct NzPrefix { int v[257]; };
__global__ void classify_cells_kernel(const __grid_constant__ CubeDesc c, const __grid_constant__ NzPrefix nz,
                                      float vmin, float scale, long long n_slots) {
    for (long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x; e < n_slots;
         e += (long long)gridDim.x * blockDim.x) {
        const long long word = e >> 5;
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
        if ((e & 31) == 0) c.cell_bits[word] = bits;
    }
}

struct HalfTable { float4 v[128]; };
__global__ void upload_half_kernel(float4* dst, const __grid_constant__ HalfTable h, int offset) {
    if (threadIdx.x < 128) dst[offset + threadIdx.x] = h.v[threadIdx.x];
}

}  // namespace

cudaError_t launch_render_global(const CubeDesc& c, const ViewDesc& v, const TFDesc& t, const RenderArgs& a, cudaStream_t s) {
    dim3 grid((v.W + kTileW - 1) / kTileW, (v.H + kTileH - 1) / kTileH);
    const bool mip = a.mode == VR_MODE_MIP;
    if (a.variant == 0) {
        if (mip) render_global_kernel<VR_MODE_MIP, 0><<<grid, kThreads, 0, s>>>(c, v, t, a);
        else render_global_kernel<VR_MODE_EA, 0><<<grid, kThreads, 0, s>>>(c, v, t, a);
    } else {
        if (mip) render_global_kernel<VR_MODE_MIP, 1><<<grid, kThreads, 0, s>>>(c, v, t, a);
        else render_global_kernel<VR_MODE_EA, 1><<<grid, kThreads, 0, s>>>(c, v, t, a);
    }
    return cudaGetLastError();
}

cudaError_t launch_render_bricks(const CubeDesc& c, const ViewDesc& v, const TFDesc& t, const RenderArgs& a,
                                 const PartialDev* d_partials, int n, int total_tiles, cudaStream_t s) {
    if (n == 0 || total_tiles == 0) return cudaSuccess;
    const bool mip = a.mode == VR_MODE_MIP;
    if (a.variant == 2) {
        if (mip) render_bricks_sp_kernel<VR_MODE_MIP><<<total_tiles, kThreads, 0, s>>>(c, v, t, a, d_partials, n);
        else render_bricks_sp_kernel<VR_MODE_EA><<<total_tiles, kThreads, 0, s>>>(c, v, t, a, d_partials, n);
    } else if (a.variant == 0) {
        if (mip) render_bricks_kernel<VR_MODE_MIP, 0><<<total_tiles, kThreads, 0, s>>>(c, v, t, a, d_partials, n);
        else render_bricks_kernel<VR_MODE_EA, 0><<<total_tiles, kThreads, 0, s>>>(c, v, t, a, d_partials, n);
    } else {
        if (mip) render_bricks_kernel<VR_MODE_MIP, 1><<<total_tiles, kThreads, 0, s>>>(c, v, t, a, d_partials, n);
        else render_bricks_kernel<VR_MODE_EA, 1><<<total_tiles, kThreads, 0, s>>>(c, v, t, a, d_partials, n);
    }
    return cudaGetLastError();
}

cudaError_t launch_classify_cells(const CubeDesc& c, const int nz_prefix[257], float vmin, float scale, cudaStream_t s) {
    NzPrefix nz;
    for (int i = 0; i < 257; ++i) nz.v[i] = nz_prefix[i];
    const long long n_slots = (long long)c.nbricks * c.cell_words_per_brick * 32;
    long long blocks = (n_slots + 255) / 256;
    if (blocks > 148LL * 32) blocks = 148LL * 32;
    classify_cells_kernel<<<(int)blocks, 256, 0, s>>>(c, nz, vmin, scale, n_slots);
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
