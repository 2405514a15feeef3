// f32 instantiations of the shared-memory-resident CG (wilson_resident.cuh); own translation unit.
#include "wilson_resident.cuh"
namespace wd {
cudaError_t launch_cg_resident_f32(const ResidentArgs &a) { return launch_cg_resident_any<float>(a); }
}  // namespace wd
