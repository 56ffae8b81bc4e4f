// S0 "cube residency" kernels (BASELINE.json north_star (2) "brick-major voxel
// layout, per-brick min/max" and (4) "a device-side generator for the synthetic cubes"):
// rebrick a linear cube, generate the synthetic cube in place, per-cell / per-brick min-max.
#include <cuda_fp16.h>

#include "vr_internal.cuh"

namespace vr {

namespace {

struct Elem { int b[3]; int l[3]; int g[3]; bool stored; bool in_cube; };

// Stored voxel i of the brick-major cube: float32, or float16 rounded to nearest even (CubeDesc::vtype).
__device__ __forceinline__ float put_voxel(const CubeDesc& c, void* cube, long long i, float v) {
    if (c.vtype == 1) { const __half h = __float2half_rn(v); reinterpret_cast<__half*>(cube)[i] = h; return __half2float(h); }
    reinterpret_cast<float*>(cube)[i] = v;
    return v;
}
__device__ __forceinline__ float get_voxel(const CubeDesc& c, long long i) {
    return c.vtype == 1 ? __half2float(__ldg(reinterpret_cast<const __half*>(c.cube) + i)) : __ldg(c.cube + i);
}

// Decompose a storage slot (brick, offset inside the brick) of the brick-major cube.
__device__ __forceinline__ Elem decode(const CubeDesc& c, long long brick, long long rem) {
    Elem e;
    int bi = (int)brick;
    e.b[0] = bi % c.G[0]; e.b[1] = (bi / c.G[0]) % c.G[1]; e.b[2] = bi / (c.G[0] * c.G[1]);
    if (c.layout == 0) {
        e.l[0] = (int)(rem % c.P[0]); long long r2 = rem / c.P[0];
        e.l[1] = (int)(r2 % c.P[1]); e.l[2] = (int)(r2 / c.P[1]);
        e.stored = e.l[2] < c.P[2];
    } else {
        const int w = (int)(rem & 31);
        long long blk = rem >> 5;
        const int tx = (int)(blk % c.T[0]); blk /= c.T[0];
        const int ty = (int)(blk % c.T[1]), tz = (int)(blk / c.T[1]);
        e.l[0] = 4 * tx + (w & 3); e.l[1] = 4 * ty + 2 * (w >> 4) + ((w >> 2) & 1); e.l[2] = 2 * tz + ((w >> 3) & 1);
        e.stored = tz < c.T[2];                       // padding slots are stored too (as zeros)
    }
    e.in_cube = e.stored;
    for (int a = 0; a < 3; ++a) {
        e.g[a] = e.b[a] * c.B[a] + e.l[a];
        if (e.l[a] > c.B[a] || e.g[a] >= c.N[a]) e.in_cube = false;
    }
    return e;
}

// slots iterated per brick by the kernels below
__host__ __device__ inline long long slots_per_brick(const CubeDesc& c) {
    return c.layout == 0 ? (long long)c.P[0] * c.P[1] * c.P[2] : c.stride;
}

// One thread per SOURCE voxel of the slab [z0, z1): the voxel goes to its own brick and, where it lies on a
// brick's first plane along an axis, also to the halo plane of the brick before it (up to 8 copies).
__global__ void rebrick_kernel(CubeDesc c, float* __restrict__ cube, const float* __restrict__ src,
                               int z0, long long n_elems, unsigned long long* __restrict__ n_bad) {
    for (long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x; e < n_elems;
         e += (long long)gridDim.x * blockDim.x) {
        const int x = (int)(e % c.N[0]);
        const long long r2 = e / c.N[0];
        const int g[3] = {x, (int)(r2 % c.N[1]), z0 + (int)(r2 / c.N[1])};
        const float v = src[e];
        // NaN / inf voxels (also: beyond the float16 range when stored as such) are refused by vr_upload_cube (rare path)
        if (!isfinite(v) || (c.vtype == 1 && !isfinite(__half2float(__float2half_rn(v))))) atomicAdd(n_bad, 1ULL);
        int b[3], l[3], nalt[3];
        for (int a = 0; a < 3; ++a) {
            b[a] = c.sh[a] >= 0 ? (g[a] >> c.sh[a]) : (g[a] / c.B[a]);
            l[a] = g[a] - b[a] * c.B[a];
            nalt[a] = (l[a] == 0 && b[a] > 0) ? 2 : 1;     // also the +1 halo plane of the previous brick
        }
        for (int hz = 0; hz < nalt[2]; ++hz)
            for (int hy = 0; hy < nalt[1]; ++hy)
                for (int hx = 0; hx < nalt[0]; ++hx) {
                    const int bx = b[0] - hx, by = b[1] - hy, bz = b[2] - hz;
                    const long long brick = bx + (long long)c.G[0] * (by + (long long)c.G[1] * bz);
                    if (brick < c.win_lo || brick >= c.win_hi) continue;
                    put_voxel(c, cube, brick * c.stride + voxel_slot(c, hx ? c.B[0] : l[0], hy ? c.B[1] : l[1], hz ? c.B[2] : l[2]), v);
                }
    }
}

__global__ void unbrick_kernel(CubeDesc c, int brick, float* __restrict__ dst, int ex, int ey, int ez) {
    long long n = (long long)ex * ey * ez;
    const long long B0 = (long long)brick * c.stride;
    for (long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x; e < n;
         e += (long long)gridDim.x * blockDim.x) {
        int x = (int)(e % ex), y = (int)((e / ex) % ey), z = (int)(e / ((long long)ex * ey));
        dst[e] = get_voxel(c, B0 + voxel_slot(c, x, y, z));
    }
}

// (min,max) of every macro-cell over its voxels plus the +1 layer (O-10: halo-inclusive), clipped
// to the cube.  One thread per cell.
__global__ void cell_minmax_kernel(CubeDesc c) {
    const long long first = (long long)c.win_lo * c.cells_per_brick, ncell = (long long)c.win_hi * c.cells_per_brick;
    for (long long e = first + (long long)blockIdx.x * blockDim.x + threadIdx.x; e < ncell;
         e += (long long)gridDim.x * blockDim.x) {
        int brick = (int)(e / c.cells_per_brick), cc = (int)(e % c.cells_per_brick);
        int ci[3] = {cc % c.C[0], (cc / c.C[0]) % c.C[1], cc / (c.C[0] * c.C[1])};
        int bi[3] = {brick % c.G[0], (brick / c.G[0]) % c.G[1], brick / (c.G[0] * c.G[1])};
        int lo[3], hi[3];
        bool empty = false;
        for (int a = 0; a < 3; ++a) {
            lo[a] = ci[a] * kCell;
            hi[a] = min(lo[a] + kCell, c.B[a]);                          // inclusive: +1 layer
            hi[a] = min(hi[a], c.N[a] - 1 - bi[a] * c.B[a]);             // stay inside the cube
            if (hi[a] < lo[a]) empty = true;
        }
        float mn = INFINITY, mx = -INFINITY;
        if (!empty) {
            const float* B = c.cube + (long long)brick * c.stride;
            for (int z = lo[2]; z <= hi[2]; ++z)
                for (int y = lo[1]; y <= hi[1]; ++y)
                    for (int x = lo[0]; x <= hi[0]; ++x) {
                        float v = __ldg(B + voxel_slot(c, x, y, z)); mn = fminf(mn, v); mx = fmaxf(mx, v);
                    }
        }
        c.cell_mm[e] = make_float2(mn, mx);
    }
}

__global__ void brick_minmax_kernel(CubeDesc c) {
    __shared__ float smn[256], smx[256];
    int brick = c.win_lo + blockIdx.x;
    float mn = INFINITY, mx = -INFINITY;
    for (int i = threadIdx.x; i < c.cells_per_brick; i += blockDim.x) {
        float2 v = c.cell_mm[(long long)brick * c.cells_per_brick + i];
        mn = fminf(mn, v.x); mx = fmaxf(mx, v.y);
    }
    smn[threadIdx.x] = mn; smx[threadIdx.x] = mx;
    __syncthreads();
    for (int s = blockDim.x / 2; s > 0; s >>= 1) {
        if (threadIdx.x < s) {
            smn[threadIdx.x] = fminf(smn[threadIdx.x], smn[threadIdx.x + s]);
            smx[threadIdx.x] = fmaxf(smx[threadIdx.x], smx[threadIdx.x + s]);
        }
        __syncthreads();
    }
    if (threadIdx.x == 0) c.brick_mm[brick] = make_float2(smn[0], smx[0]);
}

// ---- synthetic cube.  Evaluated in fp64 and rounded once to float32, in the
// operation order DESIGN.md "Generator" fixes, so that the bytes do not depend on the brick size.
__device__ __forceinline__ uint64_t mix64(uint64_t z) {       // splitmix64 finaliser
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
    return z ^ (z >> 31);
}

__device__ __forceinline__ double gauss_noise(uint64_t seed, uint64_t idx) {
    uint64_t z = mix64(seed + (idx + 1ULL) * 0x9E3779B97F4A7C15ULL);
    unsigned h1 = (unsigned)(z >> 32), h2 = (unsigned)(z & 0xFFFFFFFFu);
    double u1 = ((double)(h1 >> 9) + 0.5) * (1.0 / 8388608.0);
    double u2 = ((double)(h2 >> 9) + 0.5) * (1.0 / 8388608.0);
    return sqrt(-2.0 * log(u1)) * cos(2.0 * 3.14159265358979323846 * u2);
}

__global__ void generate_kernel(CubeDesc c, float* __restrict__ cube, GenDev g, long long n_elems) {
    const long long per = slots_per_brick(c);
    for (long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x; e < n_elems;
         e += (long long)gridDim.x * blockDim.x) {
        long long brick = c.win_lo + e / per, rem = e % per;
        Elem el = decode(c, brick, rem);
        float out = 0.0f;
        if (el.in_cube) {
            const int x = el.g[0], y = el.g[1], z = el.g[2];
            const int tile = (x >> 5) + g.tiles[0] * ((y >> 5) + g.tiles[1] * (z >> 5));
            const int t0 = g.tile_offsets[tile], t1 = g.tile_offsets[tile + 1];
            bool zero = false;
            if (t0 < 0 || t1 < 0) {           // negative offsets flag tiles that meet a zero box
                for (int b = 0; b < g.n_zero && !zero; ++b) {
                    const int* Bx = g.zero_boxes + 6 * b;
                    zero = x >= Bx[0] && x <= Bx[1] && y >= Bx[2] && y <= Bx[3] && z >= Bx[4] && z <= Bx[5];
                }
            }
            if (!zero) {
                uint64_t idx = (uint64_t)x + (uint64_t)c.N[0] * ((uint64_t)y + (uint64_t)c.N[1] * (uint64_t)z);
                double v = gauss_noise(g.seed, idx);
                if (c.N[2] > 1) v += g.continuum * (double)z / (double)(c.N[2] - 1);
                const int s0 = t0 < 0 ? ~t0 : t0, s1 = t1 < 0 ? ~t1 : t1;
                for (int si = s0; si < s1; ++si) {                 // ascending source id
                    const double* P = g.sources + 16 * (long long)g.tile_ids[si];
                    if (x < P[10] || x > P[11] || y < P[12] || y > P[13] || z < P[14] || z > P[15]) continue;
                    double dx = x - P[0], dy = y - P[1];
                    double xr = P[7] * dx + P[8] * dy, yr = -P[8] * dx + P[7] * dy;
                    double zr = ((double)z - P[2] - P[9] * xr) / P[6];
                    double q = xr * xr / (P[4] * P[4]) + yr * yr / (P[5] * P[5]) + zr * zr;
                    v += P[3] * exp(-0.5 * q);
                }
                out = (float)v;
            }
        }
        if (el.stored) put_voxel(c, cube, brick * c.stride + rem, out);
    }
}

int grid_for(long long n, int threads) {
    long long b = (n + threads - 1) / threads;
    const long long cap = 148LL * 64;
    return (int)(b < 1 ? 1 : (b > cap ? cap : b));
}

}  // namespace

cudaError_t launch_rebrick(const CubeDesc& c, float* d_cube, const float* d_src, int z0, int z1, unsigned long long* d_bad,
                           cudaStream_t s) {
    const long long n = (long long)c.N[0] * c.N[1] * (z1 - z0);
    if (n <= 0) return cudaSuccess;
    rebrick_kernel<<<grid_for(n, 256), 256, 0, s>>>(c, d_cube, d_src, z0, n, d_bad);
    return cudaGetLastError();
}

cudaError_t launch_unbrick(const CubeDesc& c, int brick, float* d_dst, cudaStream_t s) {
    int bi[3] = {brick % c.G[0], (brick / c.G[0]) % c.G[1], brick / (c.G[0] * c.G[1])};
    int e[3];
    for (int a = 0; a < 3; ++a) e[a] = std::min(c.B[a], c.N[a] - bi[a] * c.B[a]);
    long long n = (long long)e[0] * e[1] * e[2];
    unbrick_kernel<<<grid_for(n, 256), 256, 0, s>>>(c, brick, d_dst, e[0], e[1], e[2]);
    return cudaGetLastError();
}

cudaError_t launch_minmax(const CubeDesc& c, cudaStream_t s) {
    long long ncell = (long long)(c.win_hi - c.win_lo) * c.cells_per_brick;
    cudaError_t e;
    if (c.layout == 1) e = launch_cell_minmax_lines(c, s);          // vr_setup.cu: whole lines, coalesced
    else { cell_minmax_kernel<<<grid_for(ncell, 128), 128, 0, s>>>(c); e = cudaGetLastError(); }
    if (e != cudaSuccess) return e;
    brick_minmax_kernel<<<c.win_hi - c.win_lo, 256, 0, s>>>(c);
    return cudaGetLastError();
}

cudaError_t launch_generate(const CubeDesc& c, float* d_cube, const GenDev& g, cudaStream_t s) {
    long long n = (long long)(c.win_hi - c.win_lo) * slots_per_brick(c);
    if (n <= 0) return cudaSuccess;
    generate_kernel<<<grid_for(n, 256), 256, 0, s>>>(c, d_cube, g, n);
    return cudaGetLastError();
}

}  // namespace vr
