// Catalogue overlay (section 2: a source finder's
// catalogue, "a set of detected astronomical sources represented by their bounding cubes ...
// superimposed as wireframe boxes on the volume rendering output"; selectable; groups shown or
// hidden).  Reading O-14: the 12 edges of every shown box are projected with the view
// matrix in fp64, clipped in clip space (w >= 1e-9, |z| <= w, guard band |x|,|y| <= 2w), mapped to
// pixel coordinates and sampled at n + 1 equidistant points, n = max(1, ceil(max(|dpx|,|dpy|))),
// each rounded to the nearest pixel.  A pixel keeps the HIGHEST id of the boxes covering it (the
// pick image), and takes that box's colour.  Every fp64 operation is a plain + - * / floor ceil
// (the library is built --fmad=false), so the pick image is reproducible bit for bit.
#include "vr_internal.cuh"

namespace vr {

namespace {

__global__ void overlay_clear_kernel(const __grid_constant__ ViewDesc V, int* __restrict__ pick) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= V.W) return;
    for (int j = blockIdx.y; j < V.H; j += gridDim.y) pick[(long long)(V.vy0 + j) * V.pitch + (V.vx0 + i)] = 0;   // gridDim.y <= 65535
}

struct Mat4 { double m[16]; };

// one thread per edge: edge = 12 * box + 4 * axis + corner
__global__ void overlay_edges_kernel(const __grid_constant__ ViewDesc V, const __grid_constant__ Mat4 M,
                                     const int* __restrict__ boxes, const unsigned char* __restrict__ visible,
                                     int n_boxes, int* __restrict__ pick) {
    const long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= 12LL * n_boxes) return;
    const int b = (int)(e / 12), a = (int)((e % 12) / 4), c = (int)(e % 4);
    if (visible && !visible[b]) return;
    const int* B = boxes + 6LL * b;
    const int a1 = (a + 1) % 3, a2 = (a + 2) % 3;
    int lo[3], hi[3];
    lo[a] = B[2 * a]; hi[a] = B[2 * a + 1];
    lo[a1] = hi[a1] = (c & 1) ? B[2 * a1 + 1] : B[2 * a1];
    lo[a2] = hi[a2] = (c & 2) ? B[2 * a2 + 1] : B[2 * a2];
    double P[2][4];
#pragma unroll
    for (int q = 0; q < 2; ++q) {
        const double x = q ? hi[0] : lo[0], y = q ? hi[1] : lo[1], z = q ? hi[2] : lo[2];
#pragma unroll
        for (int r = 0; r < 4; ++r) P[q][r] = ((M.m[4 * r] * x + M.m[4 * r + 1] * y) + M.m[4 * r + 2] * z) + M.m[4 * r + 3];
    }
    double t0 = 0.0, t1 = 1.0;
    for (int pl = 0; pl < 7; ++pl) {                          // f(P) >= 0 keeps the point
        double f[2];
#pragma unroll
        for (int q = 0; q < 2; ++q) {
            const double x = P[q][0], y = P[q][1], z = P[q][2], w = P[q][3];
            f[q] = pl == 0 ? w - 1e-9 : pl == 1 ? z + w : pl == 2 ? w - z : pl == 3 ? x + 2.0 * w :
                   pl == 4 ? 2.0 * w - x : pl == 5 ? y + 2.0 * w : 2.0 * w - y;
        }
        if (f[0] < 0.0 && f[1] < 0.0) return;
        if (f[0] < 0.0) t0 = fmax(t0, f[0] / (f[0] - f[1]));
        if (f[1] < 0.0) t1 = fmin(t1, f[0] / (f[0] - f[1]));
    }
    if (!(t0 <= t1)) return;
    double px[2], py[2];
#pragma unroll
    for (int q = 0; q < 2; ++q) {
        const double t = q ? t1 : t0;
        const double x = P[0][0] + (P[1][0] - P[0][0]) * t, y = P[0][1] + (P[1][1] - P[0][1]) * t;
        const double w = P[0][3] + (P[1][3] - P[0][3]) * t;
        px[q] = ((x / w) + 1.0) * 0.5 * (double)V.W - 0.5;
        py[q] = (1.0 - (y / w)) * 0.5 * (double)V.H - 0.5;
    }
    const double dx = px[1] - px[0], dy = py[1] - py[0];
    const double len = ceil(fmax(fabs(dx), fabs(dy)));
    if (!(len < 1.0e7)) return;
    const int ns = len < 1.0 ? 1 : (int)len;
    for (int s = 0; s <= ns; ++s) {
        const double t = (double)s / (double)ns;
        const double X = px[0] + dx * t, Y = py[0] + dy * t;
        const double fi = floor(X + 0.5), fj = floor(Y + 0.5);
        if (!(fi >= 0.0 && fi < (double)V.W && fj >= 0.0 && fj < (double)V.H)) continue;
        atomicMax(&pick[(long long)(V.vy0 + (int)fj) * V.pitch + (V.vx0 + (int)fi)], b + 1);
    }
}

__global__ void overlay_paint_kernel(const __grid_constant__ ViewDesc V, const int* __restrict__ pick,
                                     const float4* __restrict__ colours, float4* __restrict__ frame) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= V.W) return;
    for (int j = blockIdx.y; j < V.H; j += gridDim.y) {
        const long long px = (long long)(V.vy0 + j) * V.pitch + (V.vx0 + i);
        const int id = pick[px];
        if (id > 0) frame[px] = __ldg(&colours[id - 1]);
    }
}

// nearest covered pixel of the (2r+1)^2 window around (x, y); ties: the larger id.  One warp.
__global__ void overlay_pick_kernel(const __grid_constant__ ViewDesc V, const int* __restrict__ pick, int x, int y, int radius,
                                    int* __restrict__ out) {
    const int side = 2 * radius + 1;
    long long best = -1;                                      // (d2 << 32) | (0x7fffffff - id): smaller is better
    for (int q = threadIdx.x; q < side * side; q += 32) {
        const int dx = q % side - radius, dy = q / side - radius;
        const int i = x + dx, j = y + dy;
        if (i < 0 || j < 0 || i >= V.W || j >= V.H) continue;
        const int id = pick[(long long)(V.vy0 + j) * V.pitch + (V.vx0 + i)] - 1;
        if (id < 0) continue;
        const long long key = ((long long)(dx * dx + dy * dy) << 32) | (long long)(0x7fffffff - id);
        if (best < 0 || key < best) best = key;
    }
    for (int o = 16; o > 0; o >>= 1) {
        const long long other = __shfl_xor_sync(0xffffffffu, best, o);
        if (other >= 0 && (best < 0 || other < best)) best = other;
    }
    if (threadIdx.x == 0) *out = best < 0 ? -1 : 0x7fffffff - (int)(best & 0xffffffffLL);
}

}  // namespace

cudaError_t launch_overlay(const ViewDesc& v, const double M[16], const int* d_boxes, const float* d_colours,
                           const unsigned char* d_visible, int n, float* d_frame, int* d_pick, cudaStream_t s) {
    dim3 grid((v.W + 255) / 256, v.H < 65535 ? v.H : 65535);
    overlay_clear_kernel<<<grid, 256, 0, s>>>(v, d_pick);
    if (n > 0) {
        Mat4 m;
        for (int i = 0; i < 16; ++i) m.m[i] = M[i];
        const long long edges = 12LL * n;
        overlay_edges_kernel<<<(unsigned)((edges + 127) / 128), 128, 0, s>>>(v, m, d_boxes, d_visible, n, d_pick);
        if (d_frame) overlay_paint_kernel<<<grid, 256, 0, s>>>(v, d_pick, reinterpret_cast<const float4*>(d_colours),
                                                               reinterpret_cast<float4*>(d_frame));
    }
    return cudaGetLastError();
}

cudaError_t launch_overlay_pick(const ViewDesc& v, const int* d_pick, int x, int y, int radius, int* d_out, cudaStream_t s) {
    overlay_pick_kernel<<<1, 32, 0, s>>>(v, d_pick, x, y, radius, d_out);
    return cudaGetLastError();
}

}  // namespace vr
