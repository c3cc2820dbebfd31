// plan PERSISTENT, Bueno-Orovio-Cherry-Fenton instantiations — see resident.cuh
#include "resident_dispatch.cuh"
namespace cardiac {
cudaError_t launch_resident_bocf(const Problem& pb, const ResidentLaunch& rl, cudaStream_t s) {
  return pb.variant == V_TANHFREE ? resident_by_stencil<Model<M_BOCF, V_TANHFREE>>(pb, rl, s)
                                  : resident_by_stencil<Model<M_BOCF, V_PAPER>>(pb, rl, s);
}
}  // namespace cardiac
