// Object-order maximum-intensity projection for per-brick partial images (BASELINE.json
// north_star (2): "shared-memory or TMA staging of brick tiles with halos").
//
// MIP is order-independent (O-5: the maximum over the taken samples), so the samples of a brick need not be visited ray
// by ray.  With sparse rays (neighbouring rays several voxels apart) an image-order marcher gathers the cube as single
// 128-byte lines in no useful order; here the cube STREAMS instead: a brick is cut into tiles of 32 x 32 x 16 cells,
// a persistent CTA brings one tile after the other (with its +1 halo: 9 x 9 x 9 lines of 4 x 4 x 2 voxels, each row of 9
// lines one bulk asynchronous copy, completion on an mbarrier; two CTAs per SM, so that the copies of one run while the
// other samples) into shared memory, finds the pixels whose rays cross the tile (the tile's projected rectangle, then the exact
// interval of lattice indices whose samples fall into the tile's cells, O-3), and takes those samples from shared
// memory, 32 consecutive samples of one ray per warp step.  A (pixel, tile) maximum goes to the brick's partial image
// with one atomic max.  Every sample is the same float32 arithmetic as in the image-order marchers (O-3, O-4), every
// sample of a brick belongs to exactly one tile: the partial images are bit-identical.
//
// Rays are set up once per view pixel (fp64, O-2) by ray_setup_kernel into a buffer of 48 bytes per pixel.
#include "vr_async.cuh"
#include "vr_sample.cuh"

namespace vr {

namespace {

constexpr int kOT0 = 32, kOT1 = 32, kOT2 = 16;              // cells of a tile
constexpr int kOB0 = kOT0 / 4 + 1, kOB1 = kOT1 / 4 + 1, kOB2 = kOT2 / 2 + 1;   // its lines per axis, halo line included
constexpr int kOLines = kOB0 * kOB1 * kOB2;
constexpr int kOThreads = 512;
constexpr int kOListCap = 1024;                             // pixels per batch of one tile
constexpr size_t kOBufBytes = (size_t)kOLines * 128;

struct TileDesc {
    int part;                // index into parts
    int tl[3];               // first cell (global voxel coordinates)
    int te[3];               // cells per axis (clipped to the brick and the cube)
    int org[3];              // voxel of slot 0 of the buffer (tl rounded down to the line grid: tl itself, tiles are aligned)
    int rx0, ry0, rw, rh;    // pixels (view coordinates) whose rays may cross the tile, clipped to the brick's rectangle
};

struct Mat4 { double m[16]; };

__device__ __forceinline__ void atomic_max_float(float* addr, float v) {
    if (v >= 0.f) atomicMax(reinterpret_cast<int*>(addr), __float_as_int(v));          // orders non-negative floats, beats any negative
    else atomicMin(reinterpret_cast<unsigned*>(addr), __float_as_uint(v));            // negative floats: smaller bits = larger value
}

// ---------------------------------------------------------------------------------------------- rays, once per view
__global__ void __launch_bounds__(kThreads)
ray_setup_kernel(const __grid_constant__ CubeDesc c, const __grid_constant__ ViewDesc V, float4* __restrict__ rays) {
    int tx, ty; tile_pixel(tx, ty);
    const int i = blockIdx.x * kTileW + tx, j = blockIdx.y * kTileH + ty;
    if (i >= V.W || j >= V.H) return;
    Ray r;
    r.o[0] = r.o[1] = r.o[2] = 0.f; r.d[0] = r.d[1] = r.d[2] = 0.f; r.inv[0] = r.inv[1] = r.inv[2] = 0.f; r.margin = 0.f;
    setup_ray(V, c, i, j, r);
    float4* out = rays + 3LL * ((long long)j * V.W + i);
    out[0] = make_float4(r.o[0], r.o[1], r.o[2], r.d[0]);
    out[1] = make_float4(r.d[1], r.d[2], r.margin, __int_as_float(r.k0));
    out[2] = make_float4(r.inv[0], r.inv[1], r.inv[2], __int_as_float(r.k1));
}

__device__ __forceinline__ void load_ray(const float4* __restrict__ rays, long long pixel, float step, Ray& r) {
    const float4 a = __ldg(rays + 3 * pixel), b = __ldg(rays + 3 * pixel + 1), cc = __ldg(rays + 3 * pixel + 2);
    r.o[0] = a.x; r.o[1] = a.y; r.o[2] = a.z; r.d[0] = a.w; r.d[1] = b.x; r.d[2] = b.y; r.margin = b.z;
    r.k0 = __float_as_int(b.w); r.inv[0] = cc.x; r.inv[1] = cc.y; r.inv[2] = cc.z; r.k1 = __float_as_int(cc.w);
    r.step = step;
}

// every pixel of every partial image starts at -inf (O-8: "-inf where a brick has no sample")
__global__ void __launch_bounds__(kThreads)
fill_partials_kernel(const PartialDev* __restrict__ parts, int n_parts) {
    __shared__ PartialDev part;
    int lx, ly;
    if (locate_tile(parts, n_parts, part, lx, ly)) reinterpret_cast<float*>(part.data)[(long long)ly * part.pitch + lx] = -INFINITY;
}

// ---------------------------------------------------------------------------------------------- the tiles
constexpr int kOGroup = 8;                                  // lanes that share one ray while sampling (a tile holds 16 - 64 samples of a ray)

// Two CTAs per SM, one tile buffer each: while one CTA samples its tile the other's lines travel.  A CTA requests the
// lines of its tile, finds the rays that cross it while they travel (that needs no voxel), waits, samples.
__global__ void __launch_bounds__(kOThreads, 2)
mip_tiles_kernel(const __grid_constant__ CubeDesc c, const __grid_constant__ ViewDesc V, const __grid_constant__ Mat4 M,
                 const PartialDev* __restrict__ parts, int n_parts, int total_tiles, const float4* __restrict__ rays,
                 unsigned long long* __restrict__ counters) {
    extern __shared__ __align__(128) unsigned char smem[];
    float* tile = reinterpret_cast<float*>(smem);
    unsigned long long* full = reinterpret_cast<unsigned long long*>(smem + kOBufBytes);
    int* list = reinterpret_cast<int*>(smem + kOBufBytes + 16);                  // kOListCap x (pixel, ka, kb)
    __shared__ TileDesc desc;
    __shared__ int n_list, next_entry;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int mine = blockIdx.x < total_tiles ? (total_tiles - 1 - (int)blockIdx.x) / (int)gridDim.x + 1 : 0;
    int cur_part = 0;                                       // warp 0: the part of the last tile described (tiles come in ascending order)

    // warp 0: describe tile i of this CTA and request its lines
    auto issue = [&](int i) {
        const int w = blockIdx.x + i * gridDim.x;
        while (cur_part + 1 < n_parts && __ldg(&parts[cur_part + 1].otile0) <= w) ++cur_part;
        const PartialDev P = parts[cur_part];
        int t = w - P.otile0;
        int blo[3], ext[3], nt[3];
#pragma unroll
        for (int a = 0; a < 3; ++a) { blo[a] = P.b[a] * c.B[a]; ext[a] = min(c.B[a], c.N[a] - blo[a]); }
        nt[0] = (ext[0] + kOT0 - 1) / kOT0; nt[1] = (ext[1] + kOT1 - 1) / kOT1; nt[2] = (ext[2] + kOT2 - 1) / kOT2;
        const int tix = t % nt[0], tiy = (t / nt[0]) % nt[1], tiz = t / (nt[0] * nt[1]);
        TileDesc d;
        d.part = cur_part;
        const int to[3] = {tix * kOT0, tiy * kOT1, tiz * kOT2};                  // first cell inside the brick
        const int tsz[3] = {kOT0, kOT1, kOT2};
#pragma unroll
        for (int a = 0; a < 3; ++a) { d.tl[a] = blo[a] + to[a]; d.te[a] = min(tsz[a], ext[a] - to[a]); d.org[a] = d.tl[a]; }
        // the lines first (they take the longest): blocks [bo, bo + nb) of the brick, a row along x = nb0 contiguous lines
        const int bo[3] = {to[0] >> 2, to[1] >> 2, to[2] >> 1};
        const int nb[3] = {min(kOB0, c.T[0] - bo[0]), min(kOB1, c.T[1] - bo[1]), min(kOB2, c.T[2] - bo[2])};
        const unsigned bar = (unsigned)__cvta_generic_to_shared(full);
        const unsigned row_bytes = (unsigned)nb[0] * 128u;
        if (lane == 0) mbar_expect_tx(bar, row_bytes * (unsigned)(nb[1] * nb[2]));
        __syncwarp();
        const float* base = c.cube + (long long)P.brick * c.stride;
        const unsigned dst0 = (unsigned)__cvta_generic_to_shared(tile);
        for (int row = lane; row < nb[1] * nb[2]; row += 32) {
            const int by = row % nb[1], bz = row / nb[1];
            bulk_load(dst0 + 128u * (unsigned)(kOB0 * (by + kOB1 * bz)),
                      base + 32LL * (bo[0] + (long long)c.T[0] * ((bo[1] + by) + (long long)c.T[1] * (bo[2] + bz))), row_bytes, bar);
        }
        // screen rectangle: the 8 corners of [tl, tl + te] (every position whose floor is a cell of the tile) through M, fp64
        double xn = 0.0, yn = 0.0;
        bool behind = false;
        if (lane < 8) {
            const double p0 = d.tl[0] + ((lane & 1) ? d.te[0] : 0), p1 = d.tl[1] + ((lane & 2) ? d.te[1] : 0), p2 = d.tl[2] + ((lane & 4) ? d.te[2] : 0);
            const double X = M.m[0] * p0 + M.m[1] * p1 + M.m[2] * p2 + M.m[3], Y = M.m[4] * p0 + M.m[5] * p1 + M.m[6] * p2 + M.m[7];
            const double Wc = M.m[12] * p0 + M.m[13] * p1 + M.m[14] * p2 + M.m[15];
            behind = !(Wc > 1e-9);
            if (!behind) { xn = X / Wc; yn = Y / Wc; }
        }
        const bool any_behind = __any_sync(0xffffffffu, behind);
        double xmin = lane < 8 ? xn : 1e300, xmax = lane < 8 ? xn : -1e300, ymin = lane < 8 ? yn : 1e300, ymax = lane < 8 ? yn : -1e300;
#pragma unroll
        for (int o = 4; o > 0; o >>= 1) {
            xmin = fmin(xmin, __shfl_xor_sync(0xffffffffu, xmin, o)); xmax = fmax(xmax, __shfl_xor_sync(0xffffffffu, xmax, o));
            ymin = fmin(ymin, __shfl_xor_sync(0xffffffffu, ymin, o)); ymax = fmax(ymax, __shfl_xor_sync(0xffffffffu, ymax, o));
        }
        int x0 = P.x0, x1 = P.x0 + P.w - 1, y0 = P.y0, y1 = P.y0 + P.h - 1;
        if (!any_behind) {                                  // as the host's brick_rect: pixel centre i has xn = 2 (i + 1/2) / W - 1
            const double fx0 = floor((xmin + 1.0) * 0.5 * V.W - 0.5) - 1.0, fx1 = ceil((xmax + 1.0) * 0.5 * V.W - 0.5) + 1.0;
            const double fy0 = floor((1.0 - ymax) * 0.5 * V.H - 0.5) - 1.0, fy1 = ceil((1.0 - ymin) * 0.5 * V.H - 0.5) + 1.0;
            x0 = max(x0, (int)fmax(fmin(fx0, 1e9), -1e9)); x1 = min(x1, (int)fmax(fmin(fx1, 1e9), -1e9));
            y0 = max(y0, (int)fmax(fmin(fy0, 1e9), -1e9)); y1 = min(y1, (int)fmax(fmin(fy1, 1e9), -1e9));
        }
        d.rx0 = x0; d.ry0 = y0; d.rw = max(0, x1 - x0 + 1); d.rh = max(0, y1 - y0 + 1);
        if (lane == 0) desc = d;                            // lane 0 holds the reduced rectangle
    };

    if (threadIdx.x == 0) {
        mbar_init((unsigned)__cvta_generic_to_shared(full), 1u);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    unsigned long long n_samples = 0;
    for (int i = 0; i < mine; ++i) {
        __syncthreads();                                    // the previous tile is sampled: buffer, list, counters and descriptor are free
        if (threadIdx.x == 0) { n_list = 0; next_entry = 0; }
        if (warp == 0) issue(i);
        __syncthreads();
        const int part = desc.part, rx0 = desc.rx0, ry0 = desc.ry0, rw = desc.rw, n_pix = desc.rw * desc.rh;
        const int tl[3] = {desc.tl[0], desc.tl[1], desc.tl[2]}, te[3] = {desc.te[0], desc.te[1], desc.te[2]};
        BrickRef tb;
        tb.base = tile; tb.lo[0] = tl[0]; tb.lo[1] = tl[1]; tb.lo[2] = tl[2];
        tb.s0 = 32u * kOB0; tb.s1 = 32u * kOB0 * kOB1;
        const float rw_inv = rw > 0 ? __frcp_rn((float)rw) : 0.f;
        bool landed = false;
        for (int base = 0; base == 0 || base < n_pix; base += kOListCap) {
            // ---- lane = pixel: the exact interval of its lattice samples whose cells belong to the tile
            for (int q = base + threadIdx.x; q < min(n_pix, base + kOListCap); q += kOThreads) {
                const int py = __float2int_rz(__fmul_rn((float)q + 0.5f, rw_inv)), px = q - py * rw;
                const long long pixel = (long long)(ry0 + py) * V.W + (rx0 + px);
                Ray r;
                load_ray(rays, pixel, V.step, r);
                int ka = r.k0, kb = r.k1;
                box_interval(r, tl, te, ka, kb);
                if (ka <= kb) {
                    const int slot = atomicAdd(&n_list, 1);
                    list[3 * slot] = q; list[3 * slot + 1] = ka; list[3 * slot + 2] = kb;
                }
            }
            __syncthreads();                                // the list is complete
            if (!landed) { mbar_wait((unsigned)__cvta_generic_to_shared(full), (unsigned)(i & 1)); landed = true; }
            // ---- kOGroup lanes = one ray, lane = sample: consecutive samples from shared memory; the groups take the
            // entries as they get free
            const int n = n_list;
            const int sub = lane & (kOGroup - 1);
            const unsigned gmask = ((1u << kOGroup) - 1u) << (lane & ~(kOGroup - 1));
            const float* P_data = reinterpret_cast<const float*>(parts[part].data);
            const long long P_pitch = parts[part].pitch;
            const int P_x0 = parts[part].x0, P_y0 = parts[part].y0;
            for (;;) {
                int e = 0;
                if (sub == 0) e = atomicAdd(&next_entry, 1);
                e = __shfl_sync(gmask, e, lane & ~(kOGroup - 1));
                if (e >= n) break;
                const int q = list[3 * e], ka = list[3 * e + 1], kb = list[3 * e + 2];
                const int py = __float2int_rz(__fmul_rn((float)q + 0.5f, rw_inv)), px = q - py * rw;
                const int vx = rx0 + px, vy = ry0 + py;
                const long long pixel = (long long)vy * V.W + vx;
                const float4 ra = __ldg(rays + 3 * pixel), rb = __ldg(rays + 3 * pixel + 1);
                float m = -INFINITY;
                for (int k = ka + sub; k <= kb; k += kOGroup) {
                    const float t = __fmul_rn((float)k, V.step);
                    float p[3];
                    p[0] = __fmaf_rn(t, ra.w, ra.x); p[1] = __fmaf_rn(t, rb.x, ra.y); p[2] = __fmaf_rn(t, rb.y, ra.z);
                    float fl[3], v[8];
                    const int ix = floor_pos(p[0], fl[0]), iy = floor_pos(p[1], fl[1]), iz = floor_pos(p[2], fl[2]);
                    unsigned qq, dx, dy, dz;
                    cell_address<1>(tb, (unsigned)(ix - tb.lo[0]), (unsigned)(iy - tb.lo[1]), (unsigned)(iz - tb.lo[2]), qq, dx, dy, dz);
                    const float* s = tile + qq;
                    v[0] = s[0]; v[1] = s[dx]; v[2] = s[dy]; v[3] = s[dy + dx];
                    v[4] = s[dz]; v[5] = s[dz + dx]; v[6] = s[dz + dy]; v[7] = s[dz + dy + dx];
                    m = fmaxf(m, trilinear(v, __fsub_rn(p[0], fl[0]), __fsub_rn(p[1], fl[1]), __fsub_rn(p[2], fl[2])));
                }
#pragma unroll
                for (int o = kOGroup / 2; o > 0; o >>= 1) m = fmaxf(m, __shfl_xor_sync(gmask, m, o));
                if (sub == 0) {
                    atomic_max_float(const_cast<float*>(P_data) + (long long)(vy - P_y0) * P_pitch + (vx - P_x0), m);
                    n_samples += (unsigned long long)(kb - ka + 1);
                }
            }
            if (base + kOListCap < n_pix) {                 // another batch of pixels of this tile
                __syncthreads();
                if (threadIdx.x == 0) { n_list = 0; next_entry = 0; }
                __syncthreads();
            }
        }
    }
    if (counters) {
        count(counters, kNominal, n_samples);
        count(counters, kTaken, n_samples);
    }
}

}  // namespace

int object_tiles_of_brick(const CubeDesc& c, const int b[3]) {
    int n = 1;
    const int tsz[3] = {kOT0, kOT1, kOT2};
    for (int a = 0; a < 3; ++a) {
        const int ext = std::min(c.B[a], c.N[a] - b[a] * c.B[a]);
        if (ext <= 0) return 0;
        n *= (ext + tsz[a] - 1) / tsz[a];
    }
    return n;
}

size_t ray_buffer_bytes(int W, int H) { return (size_t)W * H * 3 * sizeof(float4); }

cudaError_t launch_mip_tiles(const CubeDesc& c, const ViewDesc& v, const double M[16], const RenderArgs& a, const PartialDev* d_partials,
                             int n, int total_pixel_tiles, int total_object_tiles, float4* d_rays, cudaStream_t s) {
    if (n == 0) return cudaSuccess;
    const size_t smem = kOBufBytes + 16 + (size_t)kOListCap * 3 * sizeof(int);
    cudaError_t e = cudaFuncSetAttribute(mip_tiles_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);   // per device
    if (e != cudaSuccess) return e;
    dim3 grid((v.W + kTileW - 1) / kTileW, (v.H + kTileH - 1) / kTileH);
    ray_setup_kernel<<<grid, kThreads, 0, s>>>(c, v, d_rays);
    if (total_pixel_tiles > 0) fill_partials_kernel<<<total_pixel_tiles, kThreads, 0, s>>>(d_partials, n);
    if (total_object_tiles > 0) {
        int dev = 0, sms = 148;
        cudaGetDevice(&dev);
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        Mat4 m;
        for (int i = 0; i < 16; ++i) m.m[i] = M[i];
        mip_tiles_kernel<<<std::min(total_object_tiles, 2 * sms), kOThreads, smem, s>>>(c, v, m, d_partials, n, total_object_tiles, d_rays, a.counters);
    }
    return cudaGetLastError();
}

}  // namespace vr
