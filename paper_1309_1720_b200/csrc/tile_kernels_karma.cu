// plan FUSED, Karma instantiations — see tile.cuh
#include "tile_dispatch.cuh"
namespace cardiac {
cudaError_t launch_fused_karma(const Problem& pb, const TileLaunch& tl, cudaStream_t s) {
  return pb.variant == V_TANHFREE ? fused_by_stencil<Model<M_KARMA, V_TANHFREE>>(pb, tl, s)
                                  : fused_by_stencil<Model<M_KARMA, V_PAPER>>(pb, tl, s);
}
}  // namespace cardiac
