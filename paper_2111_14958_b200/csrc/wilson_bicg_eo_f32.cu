// fp32 instantiations of the BiCGSTAB stencil modes (MODE_RV, MODE_TS) on one parity of the lattice (even-odd
// preconditioned BiCGSTAB: SURVEY.md 8(f3) x 8(f4)); own translation unit for parallel builds.
#include "wilson_launch.cuh"
namespace wd {
cudaError_t launch_dslash_eo_bi_f32(int tile, int mode, const DslashArgs &a)
{
    if (mode == MODE_RV) return launch_dslash_tile<float, 0, MODE_RV, 18, 1>(tile, a);
    if (mode == MODE_TS) return launch_dslash_tile<float, 0, MODE_TS, 18, 1>(tile, a);
    return cudaErrorInvalidValue;
}
}  // namespace wd
