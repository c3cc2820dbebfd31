// probe_kernels.cu — diagnostic entry behind cardiac_probe(): evaluates the device-side math
// primitives (fastmath.cuh) and the pointwise reactions N[z] (models.cuh) on caller-supplied
// samples, so that tests can compare them with libm / the oracle value by value, outside any
// time stepping.  Not on the hot path.
#include "plans.h"
#include "stage.cuh"

namespace cardiac {
namespace {

__global__ void math_probe_kernel(int what, const double* __restrict__ x, double* __restrict__ out,
                                  long long n, double k) {
  const long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= n) return;
  const double v = x[e];
  out[e] = what == PROBE_EXP ? exp_c(v) : (what == PROBE_RCP ? rcp_pos(v) : hk(v, k));
}

template <class MD>
__global__ void reaction_probe_kernel(const __grid_constant__ typename MD::Params p,
                                      const double* __restrict__ z, double* __restrict__ f,
                                      long long n) {
  const long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= n) return;
  double zz[MD::NV], ff[MD::NV];
#pragma unroll
  for (int q = 0; q < MD::NV; ++q) zz[q] = z[e * MD::NV + q];
  MD::reaction(p, zz, ff);
#pragma unroll
  for (int q = 0; q < MD::NV; ++q) f[e * MD::NV + q] = ff[q];
}

template <class MD>
cudaError_t run_reaction(const Problem& pb, const double* z, double* f, long long n, cudaStream_t s) {
  typename MD::Params p;
  MD::derive(pb.params, p);
  reaction_probe_kernel<MD><<<(unsigned)((n + 127) / 128), 128, 0, s>>>(p, z, f, n);
  return cudaGetLastError();
}

}  // namespace

cudaError_t launch_probe(const Problem& pb, int what, const double* in, double* out, long long n,
                         cudaStream_t s) {
  if (n <= 0) return cudaSuccess;
  if (what == PROBE_EXP || what == PROBE_RCP || what == PROBE_HK) {
    const double k = pb.model == M_FHN ? 28.4 : (pb.model == M_KARMA ? pb.params[8] : pb.params[1]);
    math_probe_kernel<<<(unsigned)((n + 127) / 128), 128, 0, s>>>(what, in, out, n, k);
    return cudaGetLastError();
  }
  if (what != PROBE_REACTION) return cudaErrorInvalidValue;
  if (pb.model == M_FHN) return run_reaction<Model<M_FHN, V_PAPER>>(pb, in, out, n, s);
  if (pb.model == M_KARMA)
    return pb.variant == V_TANHFREE ? run_reaction<Model<M_KARMA, V_TANHFREE>>(pb, in, out, n, s)
                                    : run_reaction<Model<M_KARMA, V_PAPER>>(pb, in, out, n, s);
  if (pb.model == M_BOCF)
    return pb.variant == V_TANHFREE ? run_reaction<Model<M_BOCF, V_TANHFREE>>(pb, in, out, n, s)
                                    : run_reaction<Model<M_BOCF, V_PAPER>>(pb, in, out, n, s);
  return cudaErrorInvalidValue;
}

}  // namespace cardiac
