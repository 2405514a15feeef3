// 64-bit instantiations of the a3 pass with the y update fused in (MODE_RUPDY); own translation unit for parallel builds.
#include "wilson_launch.cuh"
namespace wd {
cudaError_t launch_dslash_y_f64(int tile, const DslashArgs &a)
{
    return launch_dslash_tile<double, 0, MODE_RUPDY>(tile, a);
}
}  // namespace wd
