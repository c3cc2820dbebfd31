// plan FUSED, Bueno-Orovio-Cherry-Fenton instantiations — see tile.cuh
#include "tile_dispatch.cuh"
namespace cardiac {
cudaError_t launch_fused_bocf(const Problem& pb, const TileLaunch& tl, cudaStream_t s) {
  return pb.variant == V_TANHFREE ? fused_by_stencil<Model<M_BOCF, V_TANHFREE>>(pb, tl, s)
                                  : fused_by_stencil<Model<M_BOCF, V_PAPER>>(pb, tl, s);
}
}  // namespace cardiac
