// B_touch (SURVEY.md 8(d) "Algorithmic bytes/flops per unit of work"): the distinct 32-byte sectors
// (and 128-byte lines) of the brick-major cube inside the 2 x 2 x 2 footprints of the samples a
// frame TAKES, i.e. interpolates after empty-space skipping (O-10) and early ray termination (O-7).
// A measurement pass for bench.py and the tests, not part of the frame path: one thread per
// (pixel, brick) walks its lattice samples one by one, applies the same exact tests as the
// marchers at the plan's skipping level, folds the taken samples (so that ERT stops where the
// marchers stop) and sets one bit per touched sector in a caller-owned bitmap.
#include "vr_sample.cuh"

namespace vr {

namespace {

__device__ __forceinline__ void mark(unsigned* __restrict__ bitmap, long long sector) {
    unsigned* w = bitmap + (sector >> 5);
    const unsigned bit = 1u << (unsigned)(sector & 31);
    if ((*(volatile unsigned*)w & bit) == 0u) atomicOr(w, bit);
}

template <int MODE, int LAYOUT, typename VT>
__global__ void __launch_bounds__(kThreads)
touch_kernel(const __grid_constant__ CubeDesc c, const __grid_constant__ ViewDesc V, const __grid_constant__ TFDesc T,
             const __grid_constant__ RenderArgs A, const PartialDev* __restrict__ parts, int n_parts,
             unsigned* __restrict__ bitmap, unsigned long long* __restrict__ n_taken) {
    __shared__ PartialDev part;
    int lx, ly;
    const bool live = locate_tile(parts, n_parts, part, lx, ly);
    Ray r; r.k0 = 0; r.k1 = -1;
    r.o[0] = r.o[1] = r.o[2] = 0.f; r.d[0] = r.d[1] = r.d[2] = 0.f; r.step = V.step; r.margin = 0.f;
    if (live) setup_ray(V, c, part.x0 + lx, part.y0 + ly, r);
    const int bid = part.brick;
    const int b[3] = {part.b[0], part.b[1], part.b[2]};
    const int lo[3] = {b[0] * c.B[0], b[1] * c.B[1], b[2] * c.B[2]};
    int ka = r.k0, kb = r.k1;
    brick_interval(c, r, b, lo, ka, kb);
    const BrickRefT<VT> br = brick_ref<LAYOUT, VT>(c, bid, lo);
    const unsigned* occ = (MODE == VR_MODE_EA && LAYOUT == 1 && A.skip >= 3) ? c.occ + (long long)bid * c.occ_words_per_brick : nullptr;
    constexpr int kShift = sizeof(VT) == 4 ? 3 : 4;                                       // voxels per 32-byte sector: 8 or 16
    const long long brick_sector0 = ((long long)(bid - c.win_lo) * c.stride) >> kShift;  // stride is a multiple of 32 voxels
    Accum acc = {{0.f, 0.f, 0.f}, 0.f, -INFINITY};
    unsigned long long taken = 0;
    bool skip_brick = false;
    if (A.skip >= 1 && MODE == VR_MODE_EA) skip_brick = __ldg(&c.brick_active[bid]) == 0;
    if (!skip_brick)
        for (int k = ka; k <= kb; ++k) {
            float p[3], fl[3];
            position(r, (float)k, p);
            const int iv[3] = {floor_pos(p[0], fl[0]), floor_pos(p[1], fl[1]), floor_pos(p[2], fl[2])};
            if (A.skip >= 1 && MODE == VR_MODE_MIP && __ldg(&c.brick_mm[bid]).y <= acc.m) break;
            if (A.skip >= 2 && cell_idle<MODE>(c, bid, lo, iv[0], iv[1], iv[2], acc.m)) continue;
            const unsigned ux = (unsigned)(iv[0] - lo[0]), uy = (unsigned)(iv[1] - lo[1]), uz = (unsigned)(iv[2] - lo[2]);
            if (occ && ((__ldg(occ + occ_word_index(c, ux, uy, uz)) >> occ_bit_index(ux, uy, uz)) & 1u) == 0u) continue;
            unsigned q, dx, dy, dz;
            cell_address<LAYOUT>(br, ux, uy, uz, q, dx, dy, dz);
            const unsigned off[8] = {q, q + dx, q + dy, q + dy + dx, q + dz, q + dz + dx, q + dz + dy, q + dz + dy + dx};
            float v[8];
#pragma unroll
            for (int e = 0; e < 8; ++e) {
                mark(bitmap, brick_sector0 + (off[e] >> kShift));
                v[e] = load_voxel(br.base + off[e]);
            }
            ++taken;
            const float val = trilinear(v, __fsub_rn(p[0], fl[0]), __fsub_rn(p[1], fl[1]), __fsub_rn(p[2], fl[2]));
            if (fold<MODE>(acc, val, T.baked, T, A.tau)) break;
        }
    count(n_taken, 0, taken);
}

__global__ void touch_count_kernel(const unsigned* __restrict__ bitmap, long long n_words, unsigned long long* __restrict__ out) {
    unsigned long long sectors = 0, lines = 0;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n_words; i += (long long)gridDim.x * blockDim.x) {
        const unsigned w = bitmap[i];
        sectors += __popc(w);
        unsigned x = w | (w >> 1);
        x |= x >> 2;
        lines += __popc(x & 0x11111111u);                   // a 128-byte line = 4 sectors = one nibble
    }
    count(out, 0, sectors);
    count(out, 1, lines);
}

}  // namespace

cudaError_t launch_touch(const CubeDesc& c, const ViewDesc& v, const TFDesc& t, const RenderArgs& a, const PartialDev* d_partials,
                         int n, int total_tiles, unsigned* d_bitmap, unsigned long long* d_taken, cudaStream_t s) {
    if (n == 0 || total_tiles == 0) return cudaSuccess;
    if (c.vtype == 1) {
        if (a.mode == VR_MODE_MIP) touch_kernel<VR_MODE_MIP, 1, __half><<<total_tiles, kThreads, 0, s>>>(c, v, t, a, d_partials, n, d_bitmap, d_taken);
        else touch_kernel<VR_MODE_EA, 1, __half><<<total_tiles, kThreads, 0, s>>>(c, v, t, a, d_partials, n, d_bitmap, d_taken);
    } else if (a.mode == VR_MODE_MIP) {
        if (c.layout == 0) touch_kernel<VR_MODE_MIP, 0, float><<<total_tiles, kThreads, 0, s>>>(c, v, t, a, d_partials, n, d_bitmap, d_taken);
        else touch_kernel<VR_MODE_MIP, 1, float><<<total_tiles, kThreads, 0, s>>>(c, v, t, a, d_partials, n, d_bitmap, d_taken);
    } else {
        if (c.layout == 0) touch_kernel<VR_MODE_EA, 0, float><<<total_tiles, kThreads, 0, s>>>(c, v, t, a, d_partials, n, d_bitmap, d_taken);
        else touch_kernel<VR_MODE_EA, 1, float><<<total_tiles, kThreads, 0, s>>>(c, v, t, a, d_partials, n, d_bitmap, d_taken);
    }
    return cudaGetLastError();
}

cudaError_t launch_touch_count(const unsigned* d_bitmap, long long n_words, unsigned long long* d_out, cudaStream_t s) {
    touch_count_kernel<<<148 * 8, 256, 0, s>>>(d_bitmap, n_words, d_out);
    return cudaGetLastError();
}

}  // namespace vr
