// The float32-voxel instantiation of the ray marchers (vr_march.cuh) and the entry points the C ABI calls.
#include "vr_march.cuh"

namespace vr {

cudaError_t launch_render_global_f16(const CubeDesc& c, const ViewDesc& v, const TFDesc& t, const RenderArgs& a, cudaStream_t s);
cudaError_t launch_render_bricks_f16(const CubeDesc& c, const ViewDesc& v, const TFDesc& t, const RenderArgs& a,
                                     const PartialDev* d_partials, int n, int total_tiles, cudaStream_t s);

cudaError_t launch_render_global(const CubeDesc& c, const ViewDesc& v, const TFDesc& t, const RenderArgs& a, cudaStream_t s) {
    return c.vtype == 1 ? launch_render_global_f16(c, v, t, a, s) : launch_render_global_t<float>(c, v, t, a, s);
}

cudaError_t launch_render_bricks(const CubeDesc& c, const ViewDesc& v, const TFDesc& t, const RenderArgs& a,
                                 const PartialDev* d_partials, int n, int total_tiles, cudaStream_t s) {
    return c.vtype == 1 ? launch_render_bricks_f16(c, v, t, a, d_partials, n, total_tiles, s)
                        : launch_render_bricks_t<float>(c, v, t, a, d_partials, n, total_tiles, s);
}

}  // namespace vr
