// fp64 instantiations of the multi-right-hand-side stencil kernel.
#include "wilson_mrhs.cuh"
namespace wd {
cudaError_t launch_mrhs_f64(int tile, int nrhs, int dagger, int mode, const MrhsArgs &a)
{
    return launch_mrhs_any<double>(tile, nrhs, dagger, mode, a);
}
}  // namespace wd
