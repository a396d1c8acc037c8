// Tiled fp32 spread / gather kernels (default path).  Placeholder: not yet enabled.
#include "kernels_common.cuh"
#include "launch.hpp"

namespace pswf {

bool fast_path_supported(const pswf_lr_plan*) { return false; }
size_t fast_record_bytes(const pswf_lr_plan*) { return 0; }
void launch_fast_prepare(pswf_lr_plan*, int, const float*, const float*, const GridGeom<float>&, cudaStream_t) {}
void launch_fast_spread(pswf_lr_plan*, int, const GridGeom<float>&, cudaStream_t) {}
void launch_fast_gather(pswf_lr_plan*, int, const GridGeom<float>&, float*, float*, cudaStream_t) {}

}  // namespace pswf
