// Output pyramid (section 3: "The rendering output is stored
// in TIFF format, which is converted to the pyramidal tiled TIFF format").  The TIFF container is
// client-side; these kernels produce its pixel content in a headless device buffer (reading O-15):
// level 0 = the float RGBA frame quantised to 8 bits, q = floor(clamp(c,0,1) * 255 + 1/2) in float32
// (product and sum rounded separately); level l+1 = 2 x 2 box reduction in integers, mean of the
// (up to 4) pixels rounded half up; levels while max(w, h) > tile; every level stored as tile x tile
// tiles, row-major over the tiles, edge tiles zero padded.
#include "vr_internal.cuh"

namespace vr {

namespace {

// tile is a power of two (checked by the API): shifts and masks, no integer division
__device__ __forceinline__ size_t tiled_index(int x, int y, int tiles_x, int tile) {
    const int sh = 31 - __clz(tile), m = tile - 1;
    return (((size_t)(y >> sh) * tiles_x + (size_t)(x >> sh)) << (2 * sh)) + ((size_t)(y & m) << sh) + (size_t)(x & m);
}

__device__ __forceinline__ unsigned quant(float c) {
    const float x = fminf(fmaxf(c, 0.f), 1.f);
    return (unsigned)floorf(__fadd_rn(__fmul_rn(x, 255.f), 0.5f));
}

// one thread per pixel of the PADDED level (tiles_x*tile x tiles_y*tile): padding is written as zero
__global__ void pyr_quantise_kernel(const float4* __restrict__ frame, long long pitch, int w, int h, int tiles_x, int tiles_y,
                                    int tile, uchar4* __restrict__ out) {
    const int x = blockIdx.x * blockDim.x + threadIdx.x;
    if (x >= tiles_x * tile) return;
    for (int y = blockIdx.y; y < tiles_y * tile; y += gridDim.y) {                   // gridDim.y <= 65535
    uchar4 q = make_uchar4(0, 0, 0, 0);
    if (x < w && y < h) {
        const float4 c = __ldg(&frame[(long long)y * pitch + x]);
        q = make_uchar4((unsigned char)quant(c.x), (unsigned char)quant(c.y), (unsigned char)quant(c.z), (unsigned char)quant(c.w));
    }
    out[tiled_index(x, y, tiles_x, tile)] = q;
    }
}

__global__ void pyr_reduce_kernel(const uchar4* __restrict__ src, int sw, int sh, int s_tiles_x, int w, int h, int tiles_x,
                                  int tiles_y, int tile, uchar4* __restrict__ out) {
    const int x = blockIdx.x * blockDim.x + threadIdx.x;
    if (x >= tiles_x * tile) return;
    for (int y = blockIdx.y; y < tiles_y * tile; y += gridDim.y) {
    uchar4 q = make_uchar4(0, 0, 0, 0);
    if (x < w && y < h) {
        unsigned s0 = 0, s1 = 0, s2 = 0, s3 = 0, n = 0;
#pragma unroll
        for (int dy = 0; dy < 2; ++dy)
#pragma unroll
            for (int dx = 0; dx < 2; ++dx) {
                const int sx = 2 * x + dx, sy = 2 * y + dy;
                if (sx < sw && sy < sh) {
                    const uchar4 p = src[tiled_index(sx, sy, s_tiles_x, tile)];
                    s0 += p.x; s1 += p.y; s2 += p.z; s3 += p.w; ++n;
                }
            }
        const unsigned r = n / 2;
        q = make_uchar4((unsigned char)((s0 + r) / n), (unsigned char)((s1 + r) / n), (unsigned char)((s2 + r) / n),
                        (unsigned char)((s3 + r) / n));
    }
    out[tiled_index(x, y, tiles_x, tile)] = q;
    }
}

}  // namespace

int pyramid_levels(int width, int height, int tile, vr_pyramid_level* lv, size_t* bytes) {
    int n = 0, w = width, h = height;
    size_t off = 0;
    for (;;) {
        if (n >= VR_PYRAMID_MAX_LEVELS) return -1;
        vr_pyramid_level& L = lv[n++];
        L.width = w; L.height = h;
        L.tiles_x = (w + tile - 1) / tile; L.tiles_y = (h + tile - 1) / tile;
        L.offset = off;
        off += (size_t)L.tiles_x * L.tiles_y * (size_t)tile * tile * 4;
        if (w <= tile && h <= tile) break;
        w = (w + 1) / 2; h = (h + 1) / 2;
    }
    *bytes = off;
    return n;
}

cudaError_t launch_pyramid(const float* d_frame, int width, int height, long long pitch, int tile, void* d_out, int* launches,
                           cudaStream_t s) {
    vr_pyramid_level lv[VR_PYRAMID_MAX_LEVELS];
    size_t bytes = 0;
    const int n = pyramid_levels(width, height, tile, lv, &bytes);
    char* base = (char*)d_out;
    for (int l = 0; l < n; ++l) {
        const vr_pyramid_level& L = lv[l];
        dim3 grid((L.tiles_x * tile + 255) / 256, L.tiles_y * tile < 65535 ? L.tiles_y * tile : 65535);
        uchar4* out = reinterpret_cast<uchar4*>(base + L.offset);
        if (l == 0) pyr_quantise_kernel<<<grid, 256, 0, s>>>(reinterpret_cast<const float4*>(d_frame), pitch, L.width, L.height, L.tiles_x,
                                                              L.tiles_y, tile, out);
        else pyr_reduce_kernel<<<grid, 256, 0, s>>>(reinterpret_cast<const uchar4*>(base + lv[l - 1].offset), lv[l - 1].width,
                                                    lv[l - 1].height, lv[l - 1].tiles_x, L.width, L.height, L.tiles_x, L.tiles_y, tile, out);
        ++*launches;
        cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) return e;
    }
    return cudaSuccess;
}

}  // namespace vr
