// f64 instantiations of the one-launch CG with the gauge field resident in shared memory (wilson_ures.cuh).
#include "wilson_ures.cuh"
namespace wd {
int ures_occupancy_f64(int row)
{
    int occ = 0;
    return ures_dispatch<double>(row, nullptr, &occ) == cudaSuccess ? occ : 0;
}
cudaError_t launch_cg_ures_f64(int row, const CgOneLaunchArgs &a) { return ures_dispatch<double>(row, &a, nullptr); }
}  // namespace wd
