// fp32 instantiations of the one-parity stencil kernel with 12-real link storage (even-odd solvers on compressed links:
// SURVEY.md 8(f3), two of its items composed); own translation unit for parallel builds.
#include "wilson_launch.cuh"
namespace wd {
cudaError_t launch_dslash12_eo_f32(int tile, int dagger, int mode, const DslashArgs &a)
{
    if (mode == MODE_RV && !dagger) return launch_dslash_tile<float, 0, MODE_RV, 12, 1>(tile, a);
    if (mode == MODE_TS && !dagger) return launch_dslash_tile<float, 0, MODE_TS, 12, 1>(tile, a);
    return launch_dslash_any<float, 12, 1>(tile, dagger, mode, a);
}
}  // namespace wd
