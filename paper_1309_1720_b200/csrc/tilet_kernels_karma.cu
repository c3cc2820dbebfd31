// plan FUSED / TMA, Karma instantiations — see tilet.cuh
#include "tilet_dispatch.cuh"
namespace cardiac {
cudaError_t launch_fusedt_karma(const Problem& pb, const TileLaunch& tl, cudaStream_t s) {
  return pb.variant == V_TANHFREE ? fusedt_by_stencil<Model<M_KARMA, V_TANHFREE>>(pb, tl, s)
                                  : fusedt_by_stencil<Model<M_KARMA, V_PAPER>>(pb, tl, s);
}
}  // namespace cardiac
