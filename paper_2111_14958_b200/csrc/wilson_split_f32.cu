// fp32 instantiations of the split one-launch CG kernel; own translation unit for parallel builds.
#include "wilson_split.cuh"
namespace wd {
cudaError_t launch_cg_split_f32(int split_tile, const CgOneLaunchArgs &a) { return launch_cg_split_any<float>(split_tile, a); }
}  // namespace wd
