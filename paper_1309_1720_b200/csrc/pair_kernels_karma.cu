// plan PAIR, Karma instantiations — see pair.cuh
#include "pair_dispatch.cuh"
namespace cardiac {
cudaError_t launch_pair_karma(const Problem& pb, const PairLaunch& pl, cudaStream_t s) {
  return pb.variant == V_TANHFREE ? pair_by_stencil<Model<M_KARMA, V_TANHFREE>>(pb, pl, s)
                                  : pair_by_stencil<Model<M_KARMA, V_PAPER>>(pb, pl, s);
}
}  // namespace cardiac
