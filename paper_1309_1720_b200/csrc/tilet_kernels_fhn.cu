// plan FUSED / TMA, FitzHugh-Nagumo instantiations — see tilet.cuh
#include "tilet_dispatch.cuh"
namespace cardiac {
cudaError_t launch_fusedt_fhn(const Problem& pb, const TileLaunch& tl, cudaStream_t s) {
  return fusedt_by_stencil<Model<M_FHN, V_PAPER>>(pb, tl, s);
}
}  // namespace cardiac
