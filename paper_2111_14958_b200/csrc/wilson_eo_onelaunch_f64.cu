// fp64 instantiations of the one-launch even-odd BiCGSTAB kernel; own translation unit for parallel builds.
#include "wilson_eo_onelaunch.cuh"
namespace wd {
cudaError_t launch_eo_bicgstab_onelaunch_f64(int tile, const EoOneLaunchArgs &a)
{
    return launch_eo_bicgstab_onelaunch_any<double>(tile, a);
}
}  // namespace wd
