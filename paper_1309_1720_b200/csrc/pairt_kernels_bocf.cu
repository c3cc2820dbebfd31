// plan PAIR / TMA, Bueno-Orovio-Cherry-Fenton instantiations — see pairt.cuh
#include "pairt_dispatch.cuh"
namespace cardiac {
cudaError_t launch_pairt_bocf(const Problem& pb, const PairTLaunch& pl, cudaStream_t s) {
  return pb.variant == V_TANHFREE ? pairt_by_stencil<Model<M_BOCF, V_TANHFREE>>(pb, pl, s)
                                  : pairt_by_stencil<Model<M_BOCF, V_PAPER>>(pb, pl, s);
}
}  // namespace cardiac
