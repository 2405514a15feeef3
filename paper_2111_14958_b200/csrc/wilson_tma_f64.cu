// f64 instantiations of the stencil kernel with the shared-memory link pipeline (wilson_tma.cuh); own translation unit.
#include "wilson_tma.cuh"
namespace wd {
cudaError_t launch_dslash_tma_f64(int row, int dagger, int mode, const TmaArgs &a)
{
    return launch_dslash_tma_any<double>(row, dagger, mode, a);
}
}  // namespace wd
