// plan PAIR, Bueno-Orovio-Cherry-Fenton instantiations — see pair.cuh
#include "pair_dispatch.cuh"
namespace cardiac {
cudaError_t launch_pair_bocf(const Problem& pb, const PairLaunch& pl, cudaStream_t s) {
  return pb.variant == V_TANHFREE ? pair_by_stencil<Model<M_BOCF, V_TANHFREE>>(pb, pl, s)
                                  : pair_by_stencil<Model<M_BOCF, V_PAPER>>(pb, pl, s);
}
}  // namespace cardiac
