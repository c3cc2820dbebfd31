// plan PERSISTENT, FitzHugh-Nagumo instantiations — see resident.cuh
#include "resident_dispatch.cuh"
namespace cardiac {
cudaError_t launch_resident_fhn(const Problem& pb, const ResidentLaunch& rl, cudaStream_t s) {
  return resident_by_stencil<Model<M_FHN, V_PAPER>>(pb, rl, s);
}
}  // namespace cardiac
