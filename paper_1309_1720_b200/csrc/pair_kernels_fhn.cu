// plan PAIR, FitzHugh-Nagumo instantiations — see pair.cuh
#include "pair_dispatch.cuh"
namespace cardiac {
cudaError_t launch_pair_fhn(const Problem& pb, const PairLaunch& pl, cudaStream_t s) {
  return pair_by_stencil<Model<M_FHN, V_PAPER>>(pb, pl, s);
}
}  // namespace cardiac
