// stage_kernels.cu — plan STAGE: one fused launch per RK substep.
//
// The paper runs (n_d + 2) kernels per substep — one Laplacian per diffusing field, one "local"
// kernel, one Euler-like update — through 2 n_s n_v global buffers and names the
// merge of these as its main optimisation direction.  Here the three are ONE
// kernel: each thread evaluates the stencil of every diffusing field, the pointwise reaction with
// the gating variables in registers, and the RK combination, and stores the next stage value.
// The kernel boundary is the paper's "lock-step" synchronisation.
#include "plans.h"
#include "stage.cuh"

namespace cardiac {

namespace {

constexpr int TX = 32, TY = 8;

template <class MD, int STENCIL, int KIND>
__global__ void __launch_bounds__(TX* TY)
    stage_direct_kernel(const __grid_constant__ StageArgs<MD> a) {
  constexpr int NV = MD::NV, ND = MD::ND;
  const int i = blockIdx.x * TX + threadIdx.x;
  const int j = blockIdx.y * TY + threadIdx.y;
  const int nx = a.g.nx, ny = a.g.ny, bc = a.g.boundary;
  if (i >= nx || j >= ny) return;
  const long long base = (long long)blockIdx.z * a.g.bstride;
  const long long row = (long long)j * a.g.pitch;
  const long long c = base + row + i;
  const double* __restrict__ in = a.in;

  double z[NV], f[NV];
#pragma unroll
  for (int q = 0; q < NV; ++q) z[q] = in[c + q * a.g.fstride];
  MD::reaction(a.p, z, f);

  // neighbour offsets with the boundary rule applied per axis (Q3)
  const long long rw1 = bidx(i - 1, nx, bc), re1 = bidx(i + 1, nx, bc);
  const long long rs1 = (long long)bidx(j - 1, ny, bc) * a.g.pitch;
  const long long rn1 = (long long)bidx(j + 1, ny, bc) * a.g.pitch;
#pragma unroll
  for (int q = 0; q < ND; ++q) {
    const double* __restrict__ U = in + base + q * a.g.fstride;
    double s;
    if (STENCIL == S_LAP5) {
      s = Stencil<S_LAP5>::apply(z[q], U[row + rw1], U[row + re1], U[rs1 + i], U[rn1 + i]);
    } else if (STENCIL == S_LAP9X4) {
      const long long rw2 = bidx(i - 2, nx, bc), re2 = bidx(i + 2, nx, bc);
      const long long rs2 = (long long)bidx(j - 2, ny, bc) * a.g.pitch;
      const long long rn2 = (long long)bidx(j + 2, ny, bc) * a.g.pitch;
      s = Stencil<S_LAP9X4>::apply(z[q], U[row + rw1], U[row + re1], U[rs1 + i], U[rn1 + i],
                                   U[row + rw2], U[row + re2], U[rs2 + i], U[rn2 + i]);
    } else {
      s = Stencil<S_BOX9>::apply(z[q], U[row + rw1], U[row + re1], U[rs1 + i], U[rn1 + i],
                                 U[rs1 + rw1], U[rs1 + re1], U[rn1 + rw1], U[rn1 + re1]);
    }
    f[q] = fma(a.lapw[q], s, f[q]);
  }

  if (KIND == K_RL || KIND == K_IE) {
    // BOCF only: u explicit Euler; gates with coefficients frozen at u^n
    if constexpr (MD::NV == 4) {
      double alpha[3], beta[3];
      MD::gates(a.p, z[0], alpha, beta);
      a.out[c] = fma(a.dt, f[0], z[0]);
#pragma unroll
      for (int g = 0; g < 3; ++g) {
        double x = z[g + 1], xn;
        if (KIND == K_RL) {
          double e = exp(alpha[g] * a.dt);
          double xinf = -beta[g] / alpha[g];
          xn = fma(x - xinf, e, xinf);
        } else {
          xn = fma(a.dt, beta[g], x) / fma(-a.dt, alpha[g], 1.0);
        }
        a.out[c + (g + 1) * a.g.fstride] = xn;
      }
    }
    return;
  }

#pragma unroll
  for (int q = 0; q < NV; ++q) {
    const long long cq = c + q * a.g.fstride;
    double yv = 0.0, Av = 0.0, Bv = 0.0;
    if (KIND != K_SELF) yv = a.y[cq];
    if (KIND == K_RK4F) { Av = a.A[cq]; Bv = a.B[cq]; }
    a.out[cq] = combine<KIND>(a.w_y, a.w_in, a.w_A, a.w_B, a.w_f, yv, z[q], Av, Bv, f[q]);
  }
}

template <class MD, int STENCIL, int KIND>
cudaError_t run(const Problem& pb, const StageLaunch& st, cudaStream_t stream) {
  StageArgs<MD> a;
  a.in = st.in; a.y = st.y; a.A = st.A; a.B = st.B; a.out = st.out;
  a.g.nx = pb.nx; a.g.ny = pb.ny; a.g.pitch = pb.pitch; a.g.boundary = pb.boundary;
  a.g.fstride = pb.fstride; a.g.bstride = pb.bstride;
  a.w_y = st.w_y; a.w_in = st.w_in; a.w_A = st.w_A; a.w_B = st.w_B; a.w_f = st.w_f;
  a.dt = pb.dt;
  MD::derive(pb.params, a.p);
  for (int q = 0; q < MD::ND; ++q) a.lapw[q] = a.p.D[q] * stencil_norm(STENCIL) / (pb.dx * pb.dx);
  dim3 grid((pb.nx + TX - 1) / TX, (pb.ny + TY - 1) / TY, pb.batch), block(TX, TY);
  stage_direct_kernel<MD, STENCIL, KIND><<<grid, block, 0, stream>>>(a);
  return cudaGetLastError();
}

template <class MD, int STENCIL>
cudaError_t by_kind(const Problem& pb, const StageLaunch& st, cudaStream_t s) {
  switch (st.kind) {
    case K_SELF: return run<MD, STENCIL, K_SELF>(pb, st, s);
    case K_BASE: return run<MD, STENCIL, K_BASE>(pb, st, s);
    case K_RK4F: return run<MD, STENCIL, K_RK4F>(pb, st, s);
    case K_RL:
      if constexpr (MD::NV == 4) return run<MD, STENCIL, K_RL>(pb, st, s);
      break;
    case K_IE:
      if constexpr (MD::NV == 4) return run<MD, STENCIL, K_IE>(pb, st, s);
      break;
  }
  return cudaErrorInvalidValue;
}

template <class MD>
cudaError_t by_stencil(const Problem& pb, const StageLaunch& st, cudaStream_t s) {
  switch (pb.stencil) {
    case S_LAP5: return by_kind<MD, S_LAP5>(pb, st, s);
    case S_LAP9X4: return by_kind<MD, S_LAP9X4>(pb, st, s);
    case S_BOX9: return by_kind<MD, S_BOX9>(pb, st, s);
  }
  return cudaErrorInvalidValue;
}

__global__ void jvp_kernel(const double* __restrict__ Z, double* __restrict__ J, int nx, int ny,
                           int nv, int pitch, long long bstride, double eps) {
  // one thread per output element of member blockIdx.z + 1
  const long long n = (long long)nx * ny * nv;
  const long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= n) return;
  const int i = (int)(e % nx);
  const long long rowf = e / nx;  // field * ny + j
  const long long src = rowf * pitch + i;
  const int b = blockIdx.y + 1;
  J[(long long)(b - 1) * n + e] = (Z[b * bstride + src] - Z[src]) / eps;
}

}  // namespace

cudaError_t launch_stage(const Problem& pb, const StageLaunch& st, cudaStream_t stream) {
  if (pb.model == M_FHN) return by_stencil<Model<M_FHN, V_PAPER>>(pb, st, stream);
  if (pb.model == M_KARMA)
    return pb.variant == V_TANHFREE ? by_stencil<Model<M_KARMA, V_TANHFREE>>(pb, st, stream)
                                    : by_stencil<Model<M_KARMA, V_PAPER>>(pb, st, stream);
  if (pb.model == M_BOCF)
    return pb.variant == V_TANHFREE ? by_stencil<Model<M_BOCF, V_TANHFREE>>(pb, st, stream)
                                    : by_stencil<Model<M_BOCF, V_PAPER>>(pb, st, stream);
  return cudaErrorInvalidValue;
}

cudaError_t launch_jvp(const Problem& pb, const double* state, double eps, double* dst,
                       cudaStream_t stream) {
  const long long n = (long long)pb.nx * pb.ny * pb.nv;
  dim3 grid((unsigned)((n + 255) / 256), pb.batch - 1);
  jvp_kernel<<<grid, 256, 0, stream>>>(state, dst, pb.nx, pb.ny, pb.nv, pb.pitch, pb.bstride, eps);
  return cudaGetLastError();
}

}  // namespace cardiac
