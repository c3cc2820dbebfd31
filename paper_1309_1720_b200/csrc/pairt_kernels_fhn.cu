// plan PAIR / TMA, FitzHugh-Nagumo instantiations — see pairt.cuh
#include "pairt_dispatch.cuh"
namespace cardiac {
cudaError_t launch_pairt_fhn(const Problem& pb, const PairTLaunch& pl, cudaStream_t s) {
  return pairt_by_stencil<Model<M_FHN, V_PAPER>>(pb, pl, s);
}
}  // namespace cardiac
