// fp64 instantiations of the stencil kernel (one translation unit per precision so that they compile in parallel).
#include "wilson_launch.cuh"
namespace wd {
cudaError_t launch_dslash_f64(int tile, int dagger, int mode, const DslashArgs &a)
{
    return launch_dslash_any<double>(tile, dagger, mode, a);
}
cudaError_t launch_cg_onelaunch_f64(int small_tile, const CgOneLaunchArgs &a)
{
    return launch_cg_onelaunch_any<double>(small_tile, a);
}
}  // namespace wd
