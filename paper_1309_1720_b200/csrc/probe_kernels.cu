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

// FP64-pipe microbenchmark: 8 independent DFMA chains per thread, registers only.  The result is
// stored so that the chains stay live; x stays bounded (|a| < 1: x -> a x + b converges).
__global__ void __launch_bounds__(256, 4) dfma_peak_kernel(double* __restrict__ sink, int iters, double a, double b) {
  double x0 = threadIdx.x * 1e-3, x1 = x0 + 0.1, x2 = x0 + 0.2, x3 = x0 + 0.3, x4 = x0 + 0.4, x5 = x0 + 0.5,
         x6 = x0 + 0.6, x7 = x0 + 0.7;
#pragma unroll 1
  for (int i = 0; i < iters; ++i) {
#pragma unroll
    for (int k = 0; k < 64; ++k) {
      x0 = fma(x0, a, b); x1 = fma(x1, a, b); x2 = fma(x2, a, b); x3 = fma(x3, a, b);
      x4 = fma(x4, a, b); x5 = fma(x5, a, b); x6 = fma(x6, a, b); x7 = fma(x7, a, b);
    }
  }
  sink[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = ((x0 + x1) + (x2 + x3)) + ((x4 + x5) + (x6 + x7));
}

// The same with M independent integer instructions (a LOP3 and an add on four separate chains) issued
// between the DFMAs of a thread's four chains: does an FP64 instruction share its issue slot?  (It does not:
// measured 2.0 / 3.7 / 6.1 cycles per DFMA and scheduler for 0 / 2 / 4 integer instructions per DFMA, i.e.
// cycles = 2 x FP64 + 1 x others — DESIGN.md "FP64 issue".)
template <int M>
__global__ void __launch_bounds__(256, 4) dfma_mix_kernel(double* __restrict__ sink, int iters, double a, double b, int ia) {
  double x0 = threadIdx.x * 1e-3, x1 = x0 + 0.1, x2 = x0 + 0.2, x3 = x0 + 0.3;
  int i0 = threadIdx.x, i1 = i0 + 1, i2 = i0 + 2, i3 = i0 + 3;
#pragma unroll 1
  for (int i = 0; i < iters; ++i) {
#pragma unroll
    for (int u = 0; u < 16; ++u) {
      x0 = fma(x0, a, b); if (M >= 1) i0 = (i0 ^ ia) + 0x1234; if (M >= 2) i1 = (i1 ^ ia) + 0x4321;
      x1 = fma(x1, a, b); if (M >= 1) i2 = (i2 ^ ia) + 0x1234; if (M >= 2) i3 = (i3 ^ ia) + 0x4321;
      x2 = fma(x2, a, b); if (M >= 1) i0 = (i0 ^ ia) + 0x1111; if (M >= 2) i1 = (i1 ^ ia) + 0x2222;
      x3 = fma(x3, a, b); if (M >= 1) i2 = (i2 ^ ia) + 0x3333; if (M >= 2) i3 = (i3 ^ ia) + 0x5555;
    }
  }
  sink[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = ((x0 + x1) + (x2 + x3)) + (double)((i0 + i1) + (i2 + i3));
}

}  // namespace

cudaError_t launch_dfma_peak(double* sink, int blocks, int iters, cudaStream_t s) {
  dfma_peak_kernel<<<blocks, kDfmaThreads, 0, s>>>(sink, iters, 0.999999, 1e-7);
  return cudaGetLastError();
}

cudaError_t launch_dfma_mix(double* sink, int blocks, int iters, int int_per_dfma, cudaStream_t s) {
  if (int_per_dfma == 0) dfma_mix_kernel<0><<<blocks, kDfmaThreads, 0, s>>>(sink, iters, 0.999999, 1e-7, 0x55);
  else if (int_per_dfma == 2) dfma_mix_kernel<1><<<blocks, kDfmaThreads, 0, s>>>(sink, iters, 0.999999, 1e-7, 0x55);
  else if (int_per_dfma == 4) dfma_mix_kernel<2><<<blocks, kDfmaThreads, 0, s>>>(sink, iters, 0.999999, 1e-7, 0x55);
  else return cudaErrorInvalidValue;
  return cudaGetLastError();
}

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
