// S5 sort-last compositing (BASELINE.json north_star (3): "an over-operator compositing kernel";
// SURVEY.md 8(a) S5, reading O-8 SORT-LAST): fold the per-brick partial images, already listed in
// visibility order, into one frame.  EA: C += (1-A) C_b, A += (1-A) A_b, then the background;
// MIP: max, then the miss value.
#include "vr_internal.cuh"

namespace vr {

namespace {

constexpr int kChunk = 2048;     // partials culled per pass against a CTA's pixel tile

template <int MODE>
__global__ void __launch_bounds__(kThreads)
composite_kernel(const __grid_constant__ ViewDesc V, const PartialDev* __restrict__ parts, int n,
                 float* __restrict__ out, float bg0, float bg1, float bg2, float bg3) {
    __shared__ unsigned mask[kChunk / 32];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int tx = (warp & 1) * 8 + (lane & 7), ty = (warp >> 1) * 4 + (lane >> 3);
    const int x0 = blockIdx.x * kTileW, y0 = blockIdx.y * kTileH;
    const int i = x0 + tx, j = y0 + ty;
    float C0 = 0.f, C1 = 0.f, C2 = 0.f, Aacc = 0.f, m = -INFINITY;
    for (int base = 0; base < n; base += kChunk) {
        const int cnt = min(kChunk, n - base);
        __syncthreads();
        if (threadIdx.x < kChunk / 32) mask[threadIdx.x] = 0u;
        __syncthreads();
        // cull: which partial rectangles of this chunk meet this CTA's pixel tile
        for (int q = threadIdx.x; q < cnt; q += kThreads) {
            const PartialDev& P = parts[base + q];
            bool hit = P.x0 < x0 + kTileW && P.x0 + P.w > x0 && P.y0 < y0 + kTileH && P.y0 + P.h > y0;
            if (hit) atomicOr(&mask[q >> 5], 1u << (q & 31));
        }
        __syncthreads();
        for (int w = 0; w < (cnt + 31) / 32; ++w) {
            unsigned bits = mask[w];
            while (bits) {                           // ascending = visibility order
                const int q = base + 32 * w + __ffs(bits) - 1;
                bits &= bits - 1;
                const PartialDev& P = parts[q];
                const int lx = i - P.x0, ly = j - P.y0;
                if (lx < 0 || ly < 0 || lx >= P.w || ly >= P.h) continue;
                const long long px = (long long)ly * P.pitch + lx;
                if (MODE == VR_MODE_MIP) {
                    m = fmaxf(m, __ldg(reinterpret_cast<const float*>(P.data) + px));
                } else {
                    const float4 pb = __ldg(reinterpret_cast<const float4*>(P.data) + px);
                    const float t = __fsub_rn(1.f, Aacc);
                    C0 = __fmaf_rn(t, pb.x, C0); C1 = __fmaf_rn(t, pb.y, C1); C2 = __fmaf_rn(t, pb.z, C2);
                    Aacc = __fmaf_rn(t, pb.w, Aacc);
                }
            }
        }
    }
    if (i < V.W && j < V.H) {
        const long long px = (long long)(V.vy0 + j) * V.pitch + (V.vx0 + i);
        if (MODE == VR_MODE_MIP) out[px] = (m == -INFINITY) ? bg0 : m;
        else {
            const float t = __fsub_rn(1.f, Aacc);
            reinterpret_cast<float4*>(out)[px] = make_float4(__fmaf_rn(t, bg0, C0), __fmaf_rn(t, bg1, C1),
                                                             __fmaf_rn(t, bg2, C2), __fmaf_rn(t, bg3, Aacc));
        }
    }
}

// NEXT-1: exchange + fold + gather of a sharded sort-last frame as ONE kernel over peer
// memory.  Every rank holds a full-frame partial image of its slab of bricks; this rank owns rows [y0, y0 + rows).
// Each thread reads its pixel from every rank's buffer (its own or a peer's mapped over NVLink: plain
// ld.global on peer pointers, no staging copy), folds the versions front to back (O-8 SORT-LAST) and stores the
// finished pixel into every rank's output frame (st.global on peer pointers: the gather).
template <int MODE>
__global__ void __launch_bounds__(128)
fold_peers_kernel(const __grid_constant__ PeerList L, int width, long long pitch, int y0, int rows, long long out_pitch,
                  float bg0, float bg1, float bg2, float bg3) {
    const long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= (long long)rows * width) return;
    const int i = (int)(e % width), j = y0 + (int)(e / width);
    const long long px = (long long)j * pitch + i;
    if (MODE == VR_MODE_MIP) {
        float m = -INFINITY;
        for (int g = 0; g < L.n; ++g) m = fmaxf(m, __ldcg(reinterpret_cast<const float*>(L.in[g]) + px));
        const float v = (m == -INFINITY) ? bg0 : m;
        for (int o = 0; o < L.n_out; ++o) reinterpret_cast<float*>(L.out[o])[(long long)j * out_pitch + i] = v;
        return;
    }
    float C0 = 0.f, C1 = 0.f, C2 = 0.f, A = 0.f;
    for (int base = 0; base < L.n; base += 8) {                // 8 peer loads in flight per thread
        float4 pb[8];
#pragma unroll
        for (int u = 0; u < 8; ++u)
            pb[u] = base + u < L.n ? __ldcg(reinterpret_cast<const float4*>(L.in[base + u]) + px) : make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            if (base + u >= L.n) break;
            const float t = __fsub_rn(1.f, A);
            C0 = __fmaf_rn(t, pb[u].x, C0); C1 = __fmaf_rn(t, pb[u].y, C1); C2 = __fmaf_rn(t, pb[u].z, C2);
            A = __fmaf_rn(t, pb[u].w, A);
        }
    }
    const float t = __fsub_rn(1.f, A);
    const float4 v = make_float4(__fmaf_rn(t, bg0, C0), __fmaf_rn(t, bg1, C1), __fmaf_rn(t, bg2, C2), __fmaf_rn(t, bg3, A));
    for (int o = 0; o < L.n_out; ++o) reinterpret_cast<float4*>(L.out[o])[(long long)j * out_pitch + i] = v;
}

}  // namespace

cudaError_t launch_fold_peers(const PeerList& L, int mode, int width, long long pitch, int y0, int rows, long long out_pitch,
                              const float bg[4], cudaStream_t s) {
    const long long n = (long long)rows * width;
    if (n <= 0) return cudaSuccess;
    const unsigned blocks = (unsigned)((n + 127) / 128);
    if (mode == VR_MODE_MIP) fold_peers_kernel<VR_MODE_MIP><<<blocks, 128, 0, s>>>(L, width, pitch, y0, rows, out_pitch, bg[0], bg[1], bg[2], bg[3]);
    else fold_peers_kernel<VR_MODE_EA><<<blocks, 128, 0, s>>>(L, width, pitch, y0, rows, out_pitch, bg[0], bg[1], bg[2], bg[3]);
    return cudaGetLastError();
}

cudaError_t launch_composite(const ViewDesc& v, int mode, const PartialDev* d_partials, int n, float* out,
                             const float bg[4], cudaStream_t s) {
    dim3 grid((v.W + kTileW - 1) / kTileW, (v.H + kTileH - 1) / kTileH);
    if (mode == VR_MODE_MIP) composite_kernel<VR_MODE_MIP><<<grid, kThreads, 0, s>>>(v, d_partials, n, out, bg[0], bg[1], bg[2], bg[3]);
    else composite_kernel<VR_MODE_EA><<<grid, kThreads, 0, s>>>(v, d_partials, n, out, bg[0], bg[1], bg[2], bg[3]);
    return cudaGetLastError();
}

}  // namespace vr
