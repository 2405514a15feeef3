// fp64 instantiations of the stencil kernel with 12-real link storage; own translation unit.
#include "wilson_launch.cuh"
namespace wd {
cudaError_t launch_dslash12_f64(int tile, int dagger, int mode, const DslashArgs &a)
{
    return launch_dslash_any<double, 12>(tile, dagger, mode, a);
}
}  // namespace wd
