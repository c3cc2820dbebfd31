// plan FUSED, FitzHugh-Nagumo instantiations — see tile.cuh
#include "tile_dispatch.cuh"
namespace cardiac {
cudaError_t launch_fused_fhn(const Problem& pb, const TileLaunch& tl, cudaStream_t s) {
  return fused_by_stencil<Model<M_FHN, V_PAPER>>(pb, tl, s);
}
}  // namespace cardiac
