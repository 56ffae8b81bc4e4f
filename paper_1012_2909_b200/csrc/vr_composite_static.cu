// S5 sort-last compositing WITHOUT any allocation (vr_composite_bricks_static, reading O-8 SORT-LAST;
// BASELINE.json north_star (3)).  vr_composite_bricks keeps the device copy of its descriptors in a buffer it allocates
// with cudaMalloc on its first call and whenever a frame has more partial images than before; callers that must not
// allocate (code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc) get this variant, whose
// descriptor scratch is a file-scope array of the library: kStaticMaxPartials descriptors, 224 KiB, held by every GPU
// that loads libvr until the process exits.
//
// The array's NAME is a host-side stand-in in host code, not a device address: the address is asked for once per device,
// with that device current (cudaGetSymbolAddress, below), and handed to the kernel as an ordinary pointer.
//
// Every call on a device shares the one array.  A call overwrites entries [0, n) before its kernel reads them and reads
// nothing beyond n, so nothing has to start at zero and stale entries of an earlier, longer call are never seen; but two
// calls whose copies / kernels overlap on the GPU (different streams, no event between them) race on it.
#include <mutex>

#include "vr_internal.cuh"

namespace vr {

namespace {

static __device__ __align__(256) unsigned char g_static_partials[(size_t)kStaticMaxPartials * sizeof(PartialDev)];

constexpr int kMaxDevices = 64;
std::mutex g_lock;
PartialDev* g_scratch[kMaxDevices] = {};     // per device: the device address of g_static_partials, asked for once

// The device address of the array on the CURRENT device (the entry point has made the context's device current).
cudaError_t static_scratch(PartialDev** out) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> hold(g_lock);
    if (!g_scratch[dev]) {
        void* p = nullptr;
        e = cudaGetSymbolAddress(&p, g_static_partials);
        if (e != cudaSuccess) return e;
        if (!p) return cudaErrorInvalidSymbol;
        g_scratch[dev] = static_cast<PartialDev*>(p);
    }
    *out = g_scratch[dev];
    return cudaSuccess;
}

constexpr int kChunk = 2048;     // partials culled per pass against a CTA's pixel tile

// composite_kernel of vr_composite.cu with its descriptors in the library's static scratch (`parts` = its device address):
// the same cull and the same fold, operation for operation, so the frames are the same to the bit.
template <int MODE>
__global__ void __launch_bounds__(kThreads)
composite_static_kernel(const __grid_constant__ ViewDesc V, const PartialDev* __restrict__ parts, int n,
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
        for (int q = threadIdx.x; q < cnt; q += kThreads) {      // cull: which rectangles of this chunk meet this CTA's tile
            const PartialDev& P = parts[base + q];
            if (P.x0 < x0 + kTileW && P.x0 + P.w > x0 && P.y0 < y0 + kTileH && P.y0 + P.h > y0) atomicOr(&mask[q >> 5], 1u << (q & 31));
        }
        __syncthreads();
        for (int w = 0; w < (cnt + 31) / 32; ++w) {
            for (unsigned bits = mask[w]; bits; bits &= bits - 1) {  // ascending = visibility order
                const PartialDev& P = parts[base + 32 * w + __ffs(bits) - 1];
                const int lx = i - P.x0, ly = j - P.y0;
                if (lx < 0 || ly < 0 || lx >= P.w || ly >= P.h) continue;
                const long long px = (long long)ly * P.pitch + lx;
                if (MODE == VR_MODE_MIP) {
                    m = fmaxf(m, __ldg(reinterpret_cast<const float*>(P.data) + px));
                } else {                                          // O-8: t = 1 - A; C = fma(t, C_b, C); A = fma(t, A_b, A)
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

}  // namespace

// Copy `count` descriptors into entries [first, first + count) of the static array of the current device (stream-ordered;
// the host buffer may be reused when the call returns: a pageable source is staged by the runtime before it does).
cudaError_t static_partials_store(int first, const PartialDev* h, int count, cudaStream_t s) {
    if (count <= 0) return cudaSuccess;
    if (first < 0 || first + count > kStaticMaxPartials) return cudaErrorInvalidValue;
    PartialDev* d = nullptr;
    cudaError_t e = static_scratch(&d);
    if (e != cudaSuccess) return e;
    return cudaMemcpyAsync(d + first, h, sizeof(PartialDev) * (size_t)count, cudaMemcpyHostToDevice, s);
}

cudaError_t launch_composite_static(const ViewDesc& v, int mode, int n, float* out, const float bg[4], cudaStream_t s) {
    if (n < 0 || n > kStaticMaxPartials) return cudaErrorInvalidValue;
    PartialDev* d = nullptr;
    cudaError_t e = static_scratch(&d);
    if (e != cudaSuccess) return e;
    dim3 grid((v.W + kTileW - 1) / kTileW, (v.H + kTileH - 1) / kTileH);
    if (mode == VR_MODE_MIP) composite_static_kernel<VR_MODE_MIP><<<grid, kThreads, 0, s>>>(v, d, n, out, bg[0], bg[1], bg[2], bg[3]);
    else composite_static_kernel<VR_MODE_EA><<<grid, kThreads, 0, s>>>(v, d, n, out, bg[0], bg[1], bg[2], bg[3]);
    return cudaGetLastError();
}

}  // namespace vr
