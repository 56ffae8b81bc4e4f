// The float16-voxel instantiation of the ray marchers (vr_march.cuh; VR_OPT_VOXEL_TYPE 1): the
// cube is stored as IEEE half precision (round to nearest even), converted back to float32 (exact) when a voxel is
// read; the arithmetic after that is the same canonical float32 as for float32 cubes.
#include "vr_march.cuh"

namespace vr {

cudaError_t launch_render_global_f16(const CubeDesc& c, const ViewDesc& v, const TFDesc& t, const RenderArgs& a, cudaStream_t s) {
    if (c.layout != 1) return cudaErrorInvalidValue;
    return launch_render_global_t<__half>(c, v, t, a, s);
}

cudaError_t launch_render_bricks_f16(const CubeDesc& c, const ViewDesc& v, const TFDesc& t, const RenderArgs& a,
                                     const PartialDev* d_partials, int n, int total_tiles, cudaStream_t s) {
    if (c.layout != 1) return cudaErrorInvalidValue;
    return launch_render_bricks_t<__half>(c, v, t, a, d_partials, n, total_tiles, s);
}

}  // namespace vr
