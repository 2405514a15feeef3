// fp64 instantiations of the BiCGSTAB stencil modes (MODE_RV, MODE_TS); own translation unit for parallel builds.
#include "wilson_launch.cuh"
namespace wd {
cudaError_t launch_dslash_bi_f64(int tile, int mode, const DslashArgs &a)
{
    if (mode == MODE_RV) return launch_dslash_tile<double, 0, MODE_RV>(tile, a);
    if (mode == MODE_TS) return launch_dslash_tile<double, 0, MODE_TS>(tile, a);
    return cudaErrorInvalidValue;
}
}  // namespace wd
