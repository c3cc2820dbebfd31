// plan PAIR / TMA, Karma instantiations — see pairt.cuh
#include "pairt_dispatch.cuh"
namespace cardiac {
cudaError_t launch_pairt_karma(const Problem& pb, const PairTLaunch& pl, cudaStream_t s) {
  return pb.variant == V_TANHFREE ? pairt_by_stencil<Model<M_KARMA, V_TANHFREE>>(pb, pl, s)
                                  : pairt_by_stencil<Model<M_KARMA, V_PAPER>>(pb, pl, s);
}
}  // namespace cardiac
