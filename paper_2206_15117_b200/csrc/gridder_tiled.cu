// gridder_tiled.cu -- tiled (output-stationary) gridding / degridding kernels.  Placeholder until the first
// measured version lands: every shape currently takes the reference path.
#include "common.cuh"

namespace imager {

bool tiled_supported(const imager_plan*) { return false; }

int launch_grid_tiled(imager_plan*, int64_t, const float2*, const float*, float2*, cudaStream_t) {
    set_error("tiled gridding not built");
    return IMAGER_ERR_UNSUPPORTED;
}

int launch_degrid_tiled(imager_plan*, int64_t, const float2*, float2*, cudaStream_t) {
    set_error("tiled degridding not built");
    return IMAGER_ERR_UNSUPPORTED;
}

}  // namespace imager
