// oracle/ovr.cpp — the CPU ORACLE.  TEST INFRASTRUCTURE ONLY (see ovr.h).
//
// Plain single-threaded ray caster: MIP and emission-absorption volume rendering of a float32
// cube under a 4x4 matrix, following, step by step, BASELINE.json `north_star` (sentences 2-3:
// "Each output pixel casts a ray ... samples it at a fixed step with trilinear interpolation, and
// either takes the maximum intensity (MIP) or maps each sample through a 256-entry RGBA transfer
// function with front-to-back emission-absorption compositing and early ray termination; the
// per-brick partial images are then composited sort-last in visibility order") and the readings
// O-1 ... O-12 of SURVEY.md section 8(c), which DESIGN.md restates.  PAPER.md gives no formula
// for any of this (line 13: "using the ray-casting algorithm").
//
// One source, instantiated twice: Real = double ("O64", the truth the tolerances are measured
// against) and Real = float ("O32", the canonical float32 arithmetic of O-11: every per-sample
// operation is one of + - * fma floor min max compare convert, IEEE-exact).  Build with
// -ffp-contract=off so that only the explicit std::fma calls below fuse.
//
// Nothing here is blocked, tiled, vectorised or reordered; there is no empty-space skipping
// (O-10: the oracle is the plain definition).  The only shortcut, the k-bracket of `bracket()`,
// is switchable (params.brute = 1 tests every lattice point) and pinned equal to brute force in
// tests/test_oracle_pins.py.
//
// Parity unpinned: anything about the paper's real cubes and figures (HIPASS, Ursa Major, the
// Duchamp catalogue) - they are not in the container (SURVEY.md 8(c) last table row).
#include "ovr.h"

#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <limits>
#include <vector>

namespace {

// ----------------------------------------------------------------------------- matrix (O-2)
bool invert4(const double a[16], double inv[16]) {      // Gauss-Jordan, partial pivoting, fp64
    double m[4][8];
    for (int r = 0; r < 4; ++r)
        for (int c = 0; c < 4; ++c) { m[r][c] = a[4 * r + c]; m[r][4 + c] = (r == c) ? 1.0 : 0.0; }
    for (int col = 0; col < 4; ++col) {
        int piv = col;
        for (int r = col + 1; r < 4; ++r) if (std::fabs(m[r][col]) > std::fabs(m[piv][col])) piv = r;
        if (m[piv][col] == 0.0) return false;
        if (piv != col) for (int c = 0; c < 8; ++c) std::swap(m[piv][c], m[col][c]);
        double p = m[col][col];
        for (int c = 0; c < 8; ++c) m[col][c] /= p;
        for (int r = 0; r < 4; ++r) {
            if (r == col) continue;
            double f = m[r][col];
            if (f != 0.0) for (int c = 0; c < 8; ++c) m[r][c] -= f * m[col][c];
        }
    }
    for (int r = 0; r < 4; ++r) for (int c = 0; c < 4; ++c) inv[4 * r + c] = m[r][4 + c];
    return true;
}

struct Camera {
    double Minv[16];
    int W, H;
    double step;
};

bool make_camera(const ovr_view* v, Camera* cam) {
    double M[16];
    for (int i = 0; i < 16; ++i) M[i] = (double)v->m[i];
    if (!invert4(M, cam->Minv)) return false;
    for (int i = 0; i < 16; ++i) if (!std::isfinite(cam->Minv[i])) return false;
    cam->W = v->width; cam->H = v->height; cam->step = (double)v->step;
    return true;
}

// Minv . (xn, yn, zn, 1), dehomogenised.  The fma nesting is part of the definition (the CUDA
// path evaluates the same expression in fp64, so both get the same bits).
void unproject(const double* Mi, double xn, double yn, double zn, double out[3]) {
    double X = std::fma(Mi[0], xn, std::fma(Mi[1], yn, std::fma(Mi[2], zn, Mi[3])));
    double Y = std::fma(Mi[4], xn, std::fma(Mi[5], yn, std::fma(Mi[6], zn, Mi[7])));
    double Z = std::fma(Mi[8], xn, std::fma(Mi[9], yn, std::fma(Mi[10], zn, Mi[11])));
    double Wc = std::fma(Mi[12], xn, std::fma(Mi[13], yn, std::fma(Mi[14], zn, Mi[15])));
    out[0] = X / Wc; out[1] = Y / Wc; out[2] = Z / Wc;
}

struct Ray64 { double o[3], d[3], L; };

// O-2: pixel (i, j), row 0 on top; o on the near plane, far point on the far plane.
Ray64 make_ray(const Camera& cam, int i, int j) {
    double xn = (2.0 * ((double)i + 0.5)) / (double)cam.W - 1.0;
    double yn = 1.0 - (2.0 * ((double)j + 0.5)) / (double)cam.H;
    double Pn[3], Pf[3];
    unproject(cam.Minv, xn, yn, -1.0, Pn);
    unproject(cam.Minv, xn, yn, +1.0, Pf);
    Ray64 r;
    double dx = Pf[0] - Pn[0], dy = Pf[1] - Pn[1], dz = Pf[2] - Pn[2];
    r.L = std::sqrt(std::fma(dx, dx, std::fma(dy, dy, dz * dz)));
    r.o[0] = Pn[0]; r.o[1] = Pn[1]; r.o[2] = Pn[2];
    r.d[0] = dx / r.L; r.d[1] = dy / r.L; r.d[2] = dz / r.L;
    return r;
}

// ----------------------------------------------------------------------------- volume (O-1)
struct Vol {
    const ovr_volume* v;
    int gx, gy, gz;
    mutable bool missing = false;
    explicit Vol(const ovr_volume* vv) : v(vv) {
        gx = (v->nx + v->bx - 1) / v->bx; gy = (v->ny + v->by - 1) / v->by; gz = (v->nz + v->bz - 1) / v->bz;
    }
    float at(int i, int j, int k) const {
        int bi = i / v->bx, bj = j / v->by, bk = k / v->bz;
        const float* B = v->bricks[bi + gx * (bj + gy * bk)];
        if (!B) { missing = true; return 0.0f; }           // the call then returns OVR_ERR_MISSING; 0 keeps the table index finite
        int ex = std::min(v->bx, v->nx - bi * v->bx), ey = std::min(v->by, v->ny - bj * v->by);
        return B[(int64_t)(i - bi * v->bx) + (int64_t)ex * ((j - bj * v->by) + (int64_t)ey * (k - bk * v->bz))];
    }
};

// ----------------------------------------------------------------------------- the marcher
template <class R> struct RayR { R o[3], d[3], L, step; };

template <class R> RayR<R> round_ray(const Ray64& r, double step) {   // O-11: rounded once
    RayR<R> q;
    for (int a = 0; a < 3; ++a) { q.o[a] = (R)r.o[a]; q.d[a] = (R)r.d[a]; }
    q.L = (R)r.L; q.step = (R)step;
    return q;
}

// O-3: t_k = k * Delta ; p_k = o + t_k d  (one fma per axis)
template <class R> inline void position(const RayR<R>& r, int64_t k, R p[3]) {
    R t = (R)k * r.step;
    for (int a = 0; a < 3; ++a) p[a] = std::fma(t, r.d[a], r.o[a]);
}

template <class R> inline bool inside(const R p[3], const int N[3]) {      // O-3 "taken"
    for (int a = 0; a < 3; ++a) if (!(p[a] >= (R)0 && p[a] <= (R)(N[a] - 1))) return false;
    return true;
}

template <class R> int64_t last_lattice_index(const RayR<R>& r) {          // largest k: t_k <= L
    int64_t k = (int64_t)std::floor((double)r.L / (double)r.step) + 2;
    while (k >= 0 && !((R)k * r.step <= r.L)) --k;
    return k;
}

// Conservative [klo, khi] containing every taken k of either precision: fp64 slab test, each slab
// widened by the float32 position error bound 2^-20 (|o_a| + L) and the result by 3 samples.  Not
// part of the definition; brute = 1 replaces it with [0, kmax].
void bracket(const Ray64& r, double step, const int N[3], int64_t kmax, int64_t* klo, int64_t* khi) {
    double t0 = 0.0, t1 = (double)kmax * step;
    for (int a = 0; a < 3; ++a) {
        double eps = (std::fabs(r.o[a]) + r.L) * (1.0 / 1048576.0);
        double lo = -eps, hi = (double)(N[a] - 1) + eps;
        if (std::fabs(r.d[a]) < 1e-9) continue;            // parallel: decided per sample
        double ta = (lo - r.o[a]) / r.d[a], tb = (hi - r.o[a]) / r.d[a];
        if (ta > tb) std::swap(ta, tb);
        t0 = std::max(t0, ta); t1 = std::min(t1, tb);
    }
    *klo = std::max<int64_t>(0, (int64_t)std::floor(t0 / step) - 3);
    *khi = std::min<int64_t>(kmax, (int64_t)std::ceil(t1 / step) + 3);
}

template <class R> inline R lerp(R a, R b, R w) { return std::fma(w, b - a, a); }   // O-4

// O-4 trilinear at p (inside the volume): x, then y, then z.
template <class R> R trilinear(const Vol& V, const R p[3], const int N[3]) {
    int i0[3], i1[3]; R w[3];
    for (int a = 0; a < 3; ++a) {
        R f = std::floor(p[a]);
        i0[a] = (int)f; w[a] = p[a] - f;
        i1[a] = std::min(i0[a] + 1, N[a] - 1);
    }
    R c000 = (R)V.at(i0[0], i0[1], i0[2]), c100 = (R)V.at(i1[0], i0[1], i0[2]);
    R c010 = (R)V.at(i0[0], i1[1], i0[2]), c110 = (R)V.at(i1[0], i1[1], i0[2]);
    R c001 = (R)V.at(i0[0], i0[1], i1[2]), c101 = (R)V.at(i1[0], i0[1], i1[2]);
    R c011 = (R)V.at(i0[0], i1[1], i1[2]), c111 = (R)V.at(i1[0], i1[1], i1[2]);
    R c00 = lerp(c000, c100, w[0]), c10 = lerp(c010, c110, w[0]);
    R c01 = lerp(c001, c101, w[0]), c11 = lerp(c011, c111, w[0]);
    R c0 = lerp(c00, c10, w[1]), c1 = lerp(c01, c11, w[1]);
    return lerp(c0, c1, w[2]);
}

// O-6 transfer function
struct BakedTF {
    float t[256][4];      // colours unchanged, alpha opacity-corrected for the step
    float vmin, vmax;
};

void bake(const ovr_tf* tf, double step, bool correct, BakedTF* b) {
    for (int i = 0; i < 256; ++i) {
        for (int c = 0; c < 3; ++c) b->t[i][c] = tf->rgba[4 * i + c];
        double a = (double)tf->rgba[4 * i + 3];
        b->t[i][3] = correct ? (float)(1.0 - std::pow(1.0 - a, step)) : (float)a;
    }
    b->vmin = tf->vmin; b->vmax = tf->vmax;
}

template <class R> void tf_lookup(const BakedTF& b, R v, R q[4]) {
    R s = (R)(255.0 / ((double)b.vmax - (double)b.vmin));
    R x = (v - (R)b.vmin) * s;
    x = std::min(std::max(x, (R)0), (R)255);
    int i = std::min((int)x, 254);
    R f = x - (R)i;
    for (int c = 0; c < 4; ++c) q[c] = lerp((R)b.t[i][c], (R)b.t[i + 1][c], f);
}

template <class R> struct Accum {          // O-5 / O-7 state of one ray (or one brick of a ray)
    R C[3] = {0, 0, 0}, A = 0, m = -std::numeric_limits<R>::infinity();
    bool stopped = false, any = false;
};

const double ERT_EDGE = 2e-5;     // O-12 knife-edge margin of the ERT decision

// One sample folded into an accumulator.  Returns true if the ray stops (ERT).
template <class R>
inline bool fold_sample(int mode, R v, const BakedTF& tf, R tau, Accum<R>& acc, bool* edge) {
    acc.any = true;
    if (mode == OVR_MIP) { acc.m = std::max(acc.m, v); return false; }
    R q[4];
    tf_lookup<R>(tf, v, q);
    R w = ((R)1 - acc.A) * q[3];                                   // O-7
    for (int c = 0; c < 3; ++c) acc.C[c] = std::fma(w, q[c], acc.C[c]);
    acc.A = acc.A + w;
    if (std::fabs((double)acc.A - (double)tau) < ERT_EDGE) *edge = true;
    if (acc.A >= tau) { acc.stopped = true; return true; }
    return false;
}

struct Keys {                       // O-9
    bool perspective;
    double eye[3];
    int sgn[3];
};

Keys view_keys(const Camera& cam, int N[3]) {
    Keys K;
    const double* Mi = cam.Minv;
    double h[4] = {Mi[2], Mi[6], Mi[10], Mi[14]};      // Minv . (0,0,1,0)^T = third column
    double nrm = std::fabs(h[0]) + std::fabs(h[1]) + std::fabs(h[2]);
    double nmax = (double)std::max(N[0], std::max(N[1], N[2]));
    K.perspective = std::fabs(h[3]) * nmax * 1e9 > nrm;
    for (int a = 0; a < 3; ++a) { K.eye[a] = 0; K.sgn[a] = 0; }
    if (K.perspective) {
        for (int a = 0; a < 3; ++a) K.eye[a] = h[a] / h[3];
    } else {
        double Pn[3], Pf[3];
        unproject(Mi, 0.0, 0.0, -1.0, Pn); unproject(Mi, 0.0, 0.0, 1.0, Pf);
        double L = std::sqrt((Pf[0]-Pn[0])*(Pf[0]-Pn[0]) + (Pf[1]-Pn[1])*(Pf[1]-Pn[1]) + (Pf[2]-Pn[2])*(Pf[2]-Pn[2]));
        for (int a = 0; a < 3; ++a) {
            double d = (Pf[a] - Pn[a]) / L;
            K.sgn[a] = d > 1e-12 ? 1 : (d < -1e-12 ? -1 : 0);
        }
    }
    return K;
}

int brick_key(const Keys& K, const int b[3], const int B[3], const int g[3]) {
    int key = 0;
    for (int a = 0; a < 3; ++a) {
        if (K.perspective) {
            int E = (int)std::floor(K.eye[a] / (double)B[a]);
            key += std::abs(b[a] - E);
        } else {
            key += K.sgn[a] > 0 ? b[a] : (K.sgn[a] < 0 ? (g[a] - 1 - b[a]) : 0);
        }
    }
    return key;
}

struct Ctx {
    Vol V;
    Camera cam;
    BakedTF tf;
    int N[3];
    explicit Ctx(const ovr_volume* v) : V(v) { N[0] = v->nx; N[1] = v->ny; N[2] = v->nz; }
};

// All taken lattice indices of one ray, in order.  The definition (O-3): k = 0, 1, ... with
// t_k <= L; taken iff the position is inside the closed box.
template <class R>
void taken_samples(const Ctx& cx, const Ray64& r64, const RayR<R>& r, bool brute,
                   std::vector<int64_t>& ks, bool* edge) {
    ks.clear();
    int64_t kmax = last_lattice_index(r);
    if (kmax < 0) return;
    int64_t klo = 0, khi = kmax;
    if (!brute) bracket(r64, cx.cam.step, cx.N, kmax, &klo, &khi);
    R p[3];
    for (int64_t k = klo; k <= khi; ++k) {
        position(r, k, p);
        if (inside(p, cx.N)) ks.push_back(k);
    }
    // O-12: the boundary-inclusion decision is a knife edge exactly when the canonical float32
    // lattice (O-11) takes a different first or last sample than this precision does.
    if (edge) {
        RayR<float> rf = round_ray<float>(r64, cx.cam.step);
        int64_t kmf = last_lattice_index(rf), f0 = -1, f1 = -1;
        float pf[3];
        for (int64_t k = std::max<int64_t>(0, klo - 1); k <= std::min(kmf, khi + 1); ++k) {
            position(rf, k, pf);
            if (inside(pf, cx.N)) { if (f0 < 0) f0 = k; f1 = k; }
        }
        int64_t g0 = ks.empty() ? -1 : ks.front(), g1 = ks.empty() ? -1 : ks.back();
        if (f0 != g0 || f1 != g1) *edge = true;
    }
}

template <class R> inline int sample_brick(const R p[3], const int PB[3], const int g[3], int b[3]) {
    for (int a = 0; a < 3; ++a) b[a] = ((int)std::floor(p[a])) / PB[a];     // O-3 membership
    return b[0] + g[0] * (b[1] + g[1] * b[2]);
}

// Render one pixel.  out: 4 floats (EA) or 1 float (MIP).
template <class R>
void render_pixel(const Ctx& cx, const ovr_params& prm, int i, int j, float* out, bool* edge,
                  ovr_counters* cnt) {
    Ray64 r64 = make_ray(cx.cam, i, j);
    RayR<R> r = round_ray<R>(r64, cx.cam.step);
    std::vector<int64_t> ks;
    taken_samples<R>(cx, r64, r, prm.brute != 0, ks, edge);
    if (cnt) cnt->nominal += (int64_t)ks.size();
    const R tau = (R)prm.tau;
    Accum<R> acc;
    R p[3];
    if (prm.split == OVR_UNSPLIT) {
        for (int64_t k : ks) {
            position(r, k, p);
            R v = trilinear<R>(cx.V, p, cx.N);
            if (cnt) cnt->taken++;
            if (fold_sample<R>(prm.mode, v, cx.tf, tau, acc, edge)) break;
        }
    } else {
        // O-8: group the taken samples by partition brick, order bricks by visibility key (O-9)
        int PB[3] = {prm.pbx, prm.pby, prm.pbz}, g[3];
        int N3[3] = {cx.N[0], cx.N[1], cx.N[2]};
        for (int a = 0; a < 3; ++a) g[a] = (cx.N[a] + PB[a] - 1) / PB[a];
        Keys K = view_keys(cx.cam, N3);
        struct Group { int key, id; std::vector<int64_t> ks; };
        std::vector<Group> groups;
        for (int64_t k : ks) {
            position(r, k, p);
            int b[3]; int id = sample_brick(p, PB, g, b);
            size_t gi = 0;
            for (; gi < groups.size(); ++gi) if (groups[gi].id == id) break;
            if (gi == groups.size()) groups.push_back({brick_key(K, b, PB, g), id, {}});
            groups[gi].ks.push_back(k);
        }
        std::stable_sort(groups.begin(), groups.end(), [](const Group& a, const Group& b) {
            return a.key != b.key ? a.key < b.key : a.id < b.id; });
        if (prm.split == OVR_SPLIT_GLOBAL) {          // one accumulator carried through bricks
            for (const Group& G : groups) {
                if (acc.stopped) break;
                for (int64_t k : G.ks) {
                    position(r, k, p);
                    R v = trilinear<R>(cx.V, p, cx.N);
                    if (cnt) cnt->taken++;
                    if (fold_sample<R>(prm.mode, v, cx.tf, tau, acc, edge)) break;
                }
            }
        } else {                                      // sort-last: per-brick partials, then fold
            for (const Group& G : groups) {
                Accum<R> pb;
                for (int64_t k : G.ks) {
                    position(r, k, p);
                    R v = trilinear<R>(cx.V, p, cx.N);
                    if (cnt) cnt->taken++;
                    if (fold_sample<R>(prm.mode, v, cx.tf, tau, pb, edge)) break;
                }
                acc.any = acc.any || pb.any;
                if (prm.mode == OVR_MIP) { acc.m = std::max(acc.m, pb.m); continue; }
                R t = (R)1 - acc.A;                   // over: frame (front) over partial (behind)
                for (int c = 0; c < 3; ++c) acc.C[c] = std::fma(t, pb.C[c], acc.C[c]);
                acc.A = std::fma(t, pb.A, acc.A);
                if (pb.stopped) acc.stopped = true;
            }
        }
    }
    if (cnt && acc.stopped) cnt->terminated++;
    if (prm.mode == OVR_MIP) {
        out[0] = acc.any ? (float)acc.m : prm.miss;
    } else {                                          // O-7: premultiplied colour over background
        R t = (R)1 - acc.A;
        for (int c = 0; c < 3; ++c) out[c] = (float)std::fma(t, (R)prm.bg[c], acc.C[c]);
        out[3] = (float)std::fma(t, (R)prm.bg[3], acc.A);
    }
}

template <class R>
void brick_pixel(const Ctx& cx, const ovr_params& prm, const int bsel[3], const int PB[3],
                 const int g[3], int i, int j, float* out) {
    Ray64 r64 = make_ray(cx.cam, i, j);
    RayR<R> r = round_ray<R>(r64, cx.cam.step);
    std::vector<int64_t> ks;
    taken_samples<R>(cx, r64, r, prm.brute != 0, ks, nullptr);
    Accum<R> acc;
    bool edge = false;
    R p[3];
    for (int64_t k : ks) {
        position(r, k, p);
        int b[3]; sample_brick(p, PB, g, b);
        if (b[0] != bsel[0] || b[1] != bsel[1] || b[2] != bsel[2]) continue;
        R v = trilinear<R>(cx.V, p, cx.N);
        if (fold_sample<R>(prm.mode, v, cx.tf, (R)prm.tau, acc, &edge)) break;
    }
    if (prm.mode == OVR_MIP) out[0] = acc.any ? (float)acc.m : -std::numeric_limits<float>::infinity();
    else { for (int c = 0; c < 3; ++c) out[c] = (float)acc.C[c]; out[3] = (float)acc.A; }
}

template <class R>
void composite_pixel(int mode, int n, const int* rects, const float* const* partials,
                     const int* order, int x, int y, const float* bg, float miss, float* out) {
    R C[3] = {0, 0, 0}, A = 0, m = -std::numeric_limits<R>::infinity();
    for (int oi = 0; oi < n; ++oi) {
        int b = order ? order[oi] : oi;
        const int* rc = rects + 4 * b;
        if (x < rc[0] || y < rc[1] || x >= rc[0] + rc[2] || y >= rc[1] + rc[3]) continue;
        size_t px = (size_t)(y - rc[1]) * rc[2] + (x - rc[0]);
        if (mode == OVR_MIP) { m = std::max(m, (R)partials[b][px]); continue; }
        const float* P = partials[b] + 4 * px;
        R t = (R)1 - A;
        for (int c = 0; c < 3; ++c) C[c] = std::fma(t, (R)P[c], C[c]);
        A = std::fma(t, (R)P[3], A);
    }
    if (mode == OVR_MIP) { out[0] = (m == -std::numeric_limits<R>::infinity()) ? miss : (float)m; return; }
    R t = (R)1 - A;
    for (int c = 0; c < 3; ++c) out[c] = (float)std::fma(t, (R)bg[c], C[c]);
    out[3] = (float)std::fma(t, (R)bg[3], A);
}

bool check_common(const ovr_volume* vol, const ovr_view* view) {
    if (!vol || !view || !vol->bricks) return false;
    if (vol->nx <= 0 || vol->ny <= 0 || vol->nz <= 0 || vol->bx <= 0 || vol->by <= 0 || vol->bz <= 0) return false;
    if (view->width <= 0 || view->height <= 0 || !(view->step > 0.0f)) return false;
    return true;
}

// splitmix64 finaliser (Steele, Lea & Flood 2014; public-domain constants), restated
inline uint64_t mix64(uint64_t z) {
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
    return z ^ (z >> 31);
}

}  // namespace

extern "C" {

int ovr_render(const ovr_volume* vol, const ovr_view* view, const ovr_tf* tf, const ovr_params* prm,
               const int* pixels, int64_t n, float* out, uint8_t* flags, ovr_counters* counters) {
    if (!check_common(vol, view) || !prm || !out) return OVR_ERR_ARG;
    if (prm->mode == OVR_EA && !tf) return OVR_ERR_ARG;
    if (tf && !(tf->vmax > tf->vmin)) return OVR_ERR_ARG;
    if (prm->split != OVR_UNSPLIT && (prm->pbx <= 0 || prm->pby <= 0 || prm->pbz <= 0)) return OVR_ERR_ARG;
    if (!pixels && n != (int64_t)view->width * view->height) return OVR_ERR_ARG;
    Ctx cx(vol);
    if (!make_camera(view, &cx.cam)) return OVR_ERR_SINGULAR;
    if (tf) bake(tf, cx.cam.step, true, &cx.tf);
    if (counters) std::memset(counters, 0, sizeof(*counters));
    const int ch = prm->mode == OVR_MIP ? 1 : 4;
    for (int64_t q = 0; q < n; ++q) {
        int i = pixels ? pixels[2 * q] : (int)(q % view->width);
        int j = pixels ? pixels[2 * q + 1] : (int)(q / view->width);
        bool edge = false;
        if (prm->precision == OVR_F32) render_pixel<float>(cx, *prm, i, j, out + ch * q, &edge, counters);
        else render_pixel<double>(cx, *prm, i, j, out + ch * q, &edge, counters);
        if (flags) flags[q] = edge ? 1 : 0;
        if (counters && edge) counters->flagged++;
    }
    return cx.V.missing ? OVR_ERR_MISSING : OVR_OK;
}

int ovr_render_brick(const ovr_volume* vol, const ovr_view* view, const ovr_tf* tf,
                     const ovr_params* prm, int brick_id, int x0, int y0, int w, int h, float* out) {
    if (!check_common(vol, view) || !prm || !out || w < 0 || h < 0) return OVR_ERR_ARG;
    if (prm->pbx <= 0 || prm->pby <= 0 || prm->pbz <= 0) return OVR_ERR_ARG;
    if (prm->mode == OVR_EA && (!tf || !(tf->vmax > tf->vmin))) return OVR_ERR_ARG;
    Ctx cx(vol);
    if (!make_camera(view, &cx.cam)) return OVR_ERR_SINGULAR;
    if (tf) bake(tf, cx.cam.step, true, &cx.tf);
    int PB[3] = {prm->pbx, prm->pby, prm->pbz}, g[3];
    for (int a = 0; a < 3; ++a) g[a] = (cx.N[a] + PB[a] - 1) / PB[a];
    if (brick_id < 0 || brick_id >= g[0] * g[1] * g[2]) return OVR_ERR_ARG;
    int bsel[3] = {brick_id % g[0], (brick_id / g[0]) % g[1], brick_id / (g[0] * g[1])};
    const int ch = prm->mode == OVR_MIP ? 1 : 4;
    for (int y = 0; y < h; ++y)
        for (int x = 0; x < w; ++x) {
            float* o = out + (size_t)ch * ((size_t)y * w + x);
            if (prm->precision == OVR_F32) brick_pixel<float>(cx, *prm, bsel, PB, g, x0 + x, y0 + y, o);
            else brick_pixel<double>(cx, *prm, bsel, PB, g, x0 + x, y0 + y, o);
        }
    return cx.V.missing ? OVR_ERR_MISSING : OVR_OK;
}

int ovr_composite(int mode, int precision, int n, const int* rects, const float* const* partials,
                  const int* order, int width, int height, const float* bg, float miss, float* out) {
    if (n < 0 || width <= 0 || height <= 0 || !out || (n > 0 && (!rects || !partials))) return OVR_ERR_ARG;
    if (mode == OVR_EA && !bg) return OVR_ERR_ARG;
    const int ch = mode == OVR_MIP ? 1 : 4;
    for (int y = 0; y < height; ++y)
        for (int x = 0; x < width; ++x) {
            float* o = out + (size_t)ch * ((size_t)y * width + x);
            if (precision == OVR_F32) composite_pixel<float>(mode, n, rects, partials, order, x, y, bg, miss, o);
            else composite_pixel<double>(mode, n, rects, partials, order, x, y, bg, miss, o);
        }
    return OVR_OK;
}

int ovr_visibility_keys(const ovr_view* view, int bx, int by, int bz, int gx, int gy, int gz,
                        int* keys, int* is_perspective) {
    if (!view || !keys || bx <= 0 || by <= 0 || bz <= 0 || gx <= 0 || gy <= 0 || gz <= 0) return OVR_ERR_ARG;
    Camera cam;
    if (!make_camera(view, &cam)) return OVR_ERR_SINGULAR;
    int N[3] = {bx * gx, by * gy, bz * gz}, B[3] = {bx, by, bz}, g[3] = {gx, gy, gz};
    Keys K = view_keys(cam, N);
    if (is_perspective) *is_perspective = K.perspective ? 1 : 0;
    for (int z = 0; z < gz; ++z) for (int y = 0; y < gy; ++y) for (int x = 0; x < gx; ++x) {
        int b[3] = {x, y, z};
        keys[x + gx * (y + gy * z)] = brick_key(K, b, B, g);
    }
    return OVR_OK;
}

int ovr_ray(const ovr_view* view, int i, int j, double o[3], double d[3], double* L) {
    if (!view || !o || !d || !L) return OVR_ERR_ARG;
    Camera cam;
    if (!make_camera(view, &cam)) return OVR_ERR_SINGULAR;
    Ray64 r = make_ray(cam, i, j);
    for (int a = 0; a < 3; ++a) { o[a] = r.o[a]; d[a] = r.d[a]; }
    *L = r.L;
    return OVR_OK;
}

int ovr_bricks_touched(const ovr_view* view, int nx, int ny, int nz, int bx, int by, int bz,
                       const int* pixels, int64_t n, uint8_t* touched) {
    if (!view || !pixels || !touched || nx <= 0 || ny <= 0 || nz <= 0 || bx <= 0 || by <= 0 || bz <= 0) return OVR_ERR_ARG;
    Camera cam;
    if (!make_camera(view, &cam)) return OVR_ERR_SINGULAR;
    int N[3] = {nx, ny, nz}, B[3] = {bx, by, bz}, g[3];
    for (int a = 0; a < 3; ++a) g[a] = (N[a] + B[a] - 1) / B[a];
    for (int64_t q = 0; q < n; ++q) {
        Ray64 r64 = make_ray(cam, pixels[2 * q], pixels[2 * q + 1]);
        RayR<double> r = round_ray<double>(r64, cam.step);
        int64_t kmax = last_lattice_index(r), klo, khi;
        if (kmax < 0) continue;
        bracket(r64, cam.step, N, kmax, &klo, &khi);
        double p[3];
        for (int64_t k = klo; k <= khi; ++k) {
            position(r, k, p);
            bool near_in = true;
            for (int a = 0; a < 3; ++a) if (!(p[a] >= -1.0 && p[a] <= N[a])) near_in = false;
            if (!near_in) continue;
            // footprint corners, one voxel of slack each way (float32 vs float64 positions)
            for (int c = 0; c < 8; ++c) {
                int b[3];
                for (int a = 0; a < 3; ++a) {
                    int v = (int)std::floor(p[a]) + (((c >> a) & 1) ? 2 : -1);
                    v = std::min(std::max(v, 0), N[a] - 1);
                    b[a] = v / B[a];
                }
                touched[b[0] + g[0] * (b[1] + g[1] * b[2])] = 1;
            }
        }
    }
    return OVR_OK;
}

int ovr_bake_tf(const ovr_tf* tf, float step, float* baked_rgba) {
    if (!tf || !baked_rgba || !(step > 0.0f)) return OVR_ERR_ARG;
    BakedTF b; bake(tf, (double)step, true, &b);
    std::memcpy(baked_rgba, b.t, sizeof(b.t));
    return OVR_OK;
}

int ovr_tf_lookup(const ovr_tf* tf, float step, int baked, double v, double rgba[4]) {
    if (!tf || !rgba || !(tf->vmax > tf->vmin)) return OVR_ERR_ARG;
    BakedTF b; bake(tf, (double)step, baked != 0, &b);
    tf_lookup<double>(b, v, rgba);
    return OVR_OK;
}

double ovr_noise(uint64_t seed, uint64_t idx) {
    // counter-based: one 64-bit hash per voxel -> two 23-bit uniforms -> Box-Muller
    uint64_t z = mix64(seed + (idx + 1) * 0x9E3779B97F4A7C15ULL);
    uint32_t h1 = (uint32_t)(z >> 32), h2 = (uint32_t)(z & 0xFFFFFFFFu);
    double u1 = ((double)(h1 >> 9) + 0.5) * (1.0 / 8388608.0);
    double u2 = ((double)(h2 >> 9) + 0.5) * (1.0 / 8388608.0);
    return std::sqrt(-2.0 * std::log(u1)) * std::cos(2.0 * 3.14159265358979323846 * u2);
}

int ovr_generate(uint64_t seed, int nx, int ny, int nz, int x0, int y0, int z0, int wx, int wy,
                 int wz, const double* S, int n_src, const int* zb, int n_zero, double continuum,
                 float* out) {
    if (nx <= 0 || ny <= 0 || nz <= 0 || wx < 0 || wy < 0 || wz < 0 || !out) return OVR_ERR_ARG;
    if (x0 < 0 || y0 < 0 || z0 < 0 || x0 + wx > nx || y0 + wy > ny || z0 + wz > nz) return OVR_ERR_ARG;
    if ((n_src > 0 && !S) || (n_zero > 0 && !zb)) return OVR_ERR_ARG;
    for (int z = z0; z < z0 + wz; ++z) for (int y = y0; y < y0 + wy; ++y) for (int x = x0; x < x0 + wx; ++x) {
        float* o = out + ((size_t)(x - x0) + (size_t)wx * ((size_t)(y - y0) + (size_t)wy * (size_t)(z - z0)));
        bool zero = false;
        for (int b = 0; b < n_zero && !zero; ++b) {
            const int* B = zb + 6 * b;
            zero = x >= B[0] && x <= B[1] && y >= B[2] && y <= B[3] && z >= B[4] && z <= B[5];
        }
        if (zero) { *o = 0.0f; continue; }
        uint64_t idx = (uint64_t)x + (uint64_t)nx * ((uint64_t)y + (uint64_t)ny * (uint64_t)z);
        double v = ovr_noise(seed, idx);
        if (nz > 1) v += continuum * (double)z / (double)(nz - 1);
        for (int s = 0; s < n_src; ++s) {                       // ascending source id
            const double* P = S + 16 * s;
            if (x < P[10] || x > P[11] || y < P[12] || y > P[13] || z < P[14] || z > P[15]) continue;
            double dx = x - P[0], dy = y - P[1];
            double xr = P[7] * dx + P[8] * dy, yr = -P[8] * dx + P[7] * dy;
            double zr = ((double)z - P[2] - P[9] * xr) / P[6];
            double q = xr * xr / (P[4] * P[4]) + yr * yr / (P[5] * P[5]) + zr * zr;
            v += P[3] * std::exp(-0.5 * q);
        }
        *o = (float)v;
    }
    return OVR_OK;
}

// ---- O-14 catalogue overlay (section 2), see ovr.h for the rule.
int ovr_overlay(const ovr_view* view, const int* boxes, int n, const uint8_t* visible, int32_t* pick) {
    if (!view || !pick || n < 0 || (n > 0 && !boxes) || view->width <= 0 || view->height <= 0) return OVR_ERR_ARG;
    const int W = view->width, H = view->height;
    for (long long i = 0; i < (long long)W * H; ++i) pick[i] = 0;
    double M[16];
    for (int i = 0; i < 16; ++i) M[i] = (double)view->m[i];
    for (int b = 0; b < n; ++b) {                            // ascending id: the highest id stays on a pixel
        if (visible && !visible[b]) continue;
        const int* B = boxes + 6 * b;
        for (int a = 0; a < 3; ++a) {                        // the 4 edges parallel to axis a
            for (int c = 0; c < 4; ++c) {
                int lo[3], hi[3];
                const int a1 = (a + 1) % 3, a2 = (a + 2) % 3;
                lo[a] = B[2 * a]; hi[a] = B[2 * a + 1];
                lo[a1] = hi[a1] = (c & 1) ? B[2 * a1 + 1] : B[2 * a1];
                lo[a2] = hi[a2] = (c & 2) ? B[2 * a2 + 1] : B[2 * a2];
                double P[2][4];                              // clip coordinates of the two ends
                for (int e = 0; e < 2; ++e) {
                    const double x = e ? hi[0] : lo[0], y = e ? hi[1] : lo[1], z = e ? hi[2] : lo[2];
                    for (int r = 0; r < 4; ++r) P[e][r] = ((M[4 * r] * x + M[4 * r + 1] * y) + M[4 * r + 2] * z) + M[4 * r + 3];
                }
                double t0 = 0.0, t1 = 1.0;
                bool out = false;
                for (int pl = 0; pl < 7 && !out; ++pl) {     // f(P) >= 0 keeps the point
                    double f[2];
                    for (int e = 0; e < 2; ++e) {
                        const double x = P[e][0], y = P[e][1], z = P[e][2], w = P[e][3];
                        switch (pl) {
                            case 0: f[e] = w - 1e-9; break;
                            case 1: f[e] = z + w; break;
                            case 2: f[e] = w - z; break;
                            case 3: f[e] = x + 2.0 * w; break;
                            case 4: f[e] = 2.0 * w - x; break;
                            case 5: f[e] = y + 2.0 * w; break;
                            default: f[e] = 2.0 * w - y; break;
                        }
                    }
                    if (f[0] < 0.0 && f[1] < 0.0) { out = true; break; }
                    if (f[0] < 0.0) t0 = std::fmax(t0, f[0] / (f[0] - f[1]));
                    if (f[1] < 0.0) t1 = std::fmin(t1, f[0] / (f[0] - f[1]));
                }
                if (out || !(t0 <= t1)) continue;
                double px[2], py[2];
                for (int e = 0; e < 2; ++e) {
                    const double t = e ? t1 : t0;
                    const double x = P[0][0] + (P[1][0] - P[0][0]) * t, y = P[0][1] + (P[1][1] - P[0][1]) * t;
                    const double w = P[0][3] + (P[1][3] - P[0][3]) * t;
                    px[e] = ((x / w) + 1.0) * 0.5 * (double)W - 0.5;
                    py[e] = (1.0 - (y / w)) * 0.5 * (double)H - 0.5;
                }
                const double dx = px[1] - px[0], dy = py[1] - py[0];
                const double len = std::ceil(std::fmax(std::fabs(dx), std::fabs(dy)));
                if (!(len < 1.0e7)) continue;                // non-finite projection
                const int ns = len < 1.0 ? 1 : (int)len;
                for (int s = 0; s <= ns; ++s) {
                    const double t = (double)s / (double)ns;
                    const double X = px[0] + dx * t, Y = py[0] + dy * t;
                    const double fi = std::floor(X + 0.5), fj = std::floor(Y + 0.5);
                    if (!(fi >= 0.0 && fi < (double)W && fj >= 0.0 && fj < (double)H)) continue;
                    int32_t& q = pick[(long long)fj * W + (long long)fi];
                    if (q < b + 1) q = b + 1;
                }
            }
        }
    }
    return OVR_OK;
}

int ovr_overlay_pick(const int32_t* pick, int width, int height, int x, int y, int radius) {
    long long best_d = -1;
    int best = -1;
    for (int dy = -radius; dy <= radius; ++dy)
        for (int dx = -radius; dx <= radius; ++dx) {
            const int i = x + dx, j = y + dy;
            if (i < 0 || j < 0 || i >= width || j >= height) continue;
            const int id = pick[(long long)j * width + i] - 1;
            if (id < 0) continue;
            const long long d = (long long)dx * dx + (long long)dy * dy;
            if (best_d < 0 || d < best_d || (d == best_d && id > best)) { best_d = d; best = id; }
        }
    return best;
}

}  // extern "C"
