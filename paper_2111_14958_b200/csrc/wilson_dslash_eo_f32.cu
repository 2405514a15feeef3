// fp32 instantiations of the stencil kernel on one parity of the lattice (even-odd).
#include "wilson_launch.cuh"
namespace wd {
cudaError_t launch_dslash_eo_f32(int tile, int dagger, int mode, const DslashArgs &a)
{
    return launch_dslash_any<float, 18, 1>(tile, dagger, mode, a);
}
}  // namespace wd
