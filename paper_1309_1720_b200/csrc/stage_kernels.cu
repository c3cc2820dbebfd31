// stage_kernels.cu — plan STAGE: one fused launch per RK substep.
//
// The paper runs (n_d + 2) kernels per substep — one Laplacian per diffusing field, one "local"
// kernel, one Euler-like update — through 2 n_s n_v global buffers and names the
// merge of these as its main optimisation direction.  Here the three are ONE
// kernel: each thread evaluates the stencil of every diffusing field, the pointwise reaction with
// the gating variables in registers, and the RK combination, and stores the next stage value.
// The kernel boundary is the paper's "lock-step" synchronisation.
//
// Layout of the work: a thread owns TWO x-adjacent cells (one 128-bit load/store per field, the
// paper's "vector width 2 for doubles"); a 32x4 block owns a 64x4 tile
// (eight blocks per SM; measured on B200 against 32x8 / 32x2: 3-10 % faster for every model from 512^2 up and in 3-D).  Blocks whose
// tile plus stencil halo lies inside the grid take a branch-free path with 128-bit neighbour loads
// served by L1; only the blocks on the rim pay for the index reflection of the no-flux boundary
// ("branching threads incur some performance penalty").
#include "plans.h"
#include "stage.cuh"

namespace cardiac {

namespace {

constexpr int TX = 32, TY = 4;   // threads; the tile is 2*TX x TY cells

// offsets inside a field: a 2-D field has fewer than 2^31 elements (checked at create), a 3-D one may not
template <bool D3> struct Off { typedef int type; };
template <> struct Off<true> { typedef long long type; };

// 3-D: the z arm of the pair (x, x+1) at offset o of a field, planes kz +- m inside the grid
template <int STENCIL>
CARDIAC_D void zarm_pair(const double* __restrict__ U, long long o, int zs, double2 c, double& s0, double& s1) {
  const double2 d1 = ld2(U + o - zs), u1 = ld2(U + o + zs);
  if (STENCIL == S_LAP9X4) {
    const double2 d2 = ld2(U + o - 2 * (long long)zs), u2 = ld2(U + o + 2 * (long long)zs);
    s0 += StencilZ<S_LAP9X4>::apply(c.x, d1.x, u1.x, d2.x, u2.x);
    s1 += StencilZ<S_LAP9X4>::apply(c.y, d1.y, u1.y, d2.y, u2.y);
  } else if (STENCIL == S_LAP5) {
    s0 += StencilZ<S_LAP5>::apply(c.x, d1.x, u1.x);
    s1 += StencilZ<S_LAP5>::apply(c.y, d1.y, u1.y);
  }
}
// ... of one cell with the boundary rule along z; oc = offset of the cell inside its plane
template <int STENCIL>
CARDIAC_D double zarm_edge(const double* __restrict__ U, int oc, int kz, int nz, int zs, int bc, double c) {
  const double d1 = U[(long long)bidx(kz - 1, nz, bc) * zs + oc], u1 = U[(long long)bidx(kz + 1, nz, bc) * zs + oc];
  if (STENCIL == S_LAP9X4) {
    const double d2 = U[(long long)bidx(kz - 2, nz, bc) * zs + oc], u2 = U[(long long)bidx(kz + 2, nz, bc) * zs + oc];
    return StencilZ<S_LAP9X4>::apply(c, d1, u1, d2, u2);
  } else if (STENCIL == S_LAP5) {
    return StencilZ<S_LAP5>::apply(c, d1, u1);
  }
  return 0.0;
}

// One gate x' = alpha x + beta with the coefficients frozen at u^n, alpha < 0:
// Rush-Larsen x+ = x_inf + (x - x_inf) e^{alpha dt}, x_inf = -beta/alpha; implicit Euler
// x+ = (x + dt beta)/(1 - dt alpha).  The division is a reciprocal of a positive number (fastmath.cuh).
template <int KIND>
CARDIAC_D double gate_step(double dt, double x, double alpha, double beta) {
  if (KIND == K_RL) {
    const double e = exp_c(alpha * dt);
    const double xinf = beta * rcp_pos(-alpha);
    return fma(x - xinf, e, xinf);
  }
  return fma(dt, beta, x) * rcp_pos(fma(-dt, alpha, 1.0));
}

// the update of one cell once f = D lap + N is known; o = offset of the cell inside its field
template <class MD, int KIND>
CARDIAC_D void finish_cell(const StageArgs<MD>& a, const double* __restrict__ yb,
                           const double* __restrict__ Ab, const double* __restrict__ Bb,
                           double* __restrict__ ob, long long o, const double (&z)[MD::NV],
                           const double (&f)[MD::NV]) {
  constexpr int NV = MD::NV;
  if (KIND == K_RL || KIND == K_IE) {
    // BOCF only: u explicit Euler; gates with coefficients frozen at u^n
    if constexpr (NV == 4) {
      double alpha[3], beta[3];
      MD::gates(a.p, z[0], alpha, beta);
      ob[o] = fma(a.dt, f[0], z[0]);
#pragma unroll
      for (int g = 0; g < 3; ++g) ob[o + (g + 1) * a.g.fstride] = gate_step<KIND>(a.dt, z[g + 1], alpha[g], beta[g]);
    }
    return;
  }
#pragma unroll
  for (int q = 0; q < NV; ++q) {
    const long long oq = o + q * a.g.fstride;
    double yv = 0.0, Av = 0.0, Bv = 0.0;
    if (KIND != K_SELF) yv = yb[oq];
    if (KIND == K_RK4F) { Av = Ab[oq]; Bv = Bb[oq]; }
    ob[oq] = combine<KIND>(a.w_y, a.w_in, a.w_A, a.w_B, a.w_f, yv, z[q], Av, Bv, f[q]);
  }
}

template <class MD, int STENCIL, int KIND, bool D3>
__global__ void __launch_bounds__(TX * TY, 8)
    stage_kernel(const __grid_constant__ StageArgs<MD> a) {
  constexpr int NV = MD::NV, ND = MD::ND;
  constexpr int R = stencil_radius(STENCIL);
  const int nx = a.g.nx, ny = a.g.ny, pitch = a.g.pitch;
  const int x0 = blockIdx.x * (2 * TX), j0 = blockIdx.y * TY;
  const int x = x0 + 2 * threadIdx.x, j = j0 + threadIdx.y;
  // 2-D: blockIdx.z = batch member.  3-D: blockIdx.z = member * nz + plane
  const int kz = D3 ? (int)(blockIdx.z % a.g.nz) : 0;
  typedef typename Off<D3>::type off_t;
  const off_t pz = D3 ? (off_t)kz * a.g.zstride : 0;            // offset of the plane inside a field
  const long long base = (long long)(D3 ? blockIdx.z / a.g.nz : blockIdx.z) * a.g.bstride;
  const double* __restrict__ in = a.in + base;
  const double* __restrict__ yb = a.y + base;
  const double* __restrict__ Ab = a.A + base;
  const double* __restrict__ Bb = a.B + base;
  double* __restrict__ ob = a.out + base;

  // block-uniform: tile and halo inside the grid -> no boundary logic, 128-bit accesses
  const bool interior = x0 >= 2 && x0 + 2 * TX + 2 <= nx && j0 >= R && j0 + TY + R <= ny &&
                        (!D3 || (kz >= R && kz + R < a.g.nz));
  const int row = j * pitch;
  const off_t o = pz + row + x;
  double2 zz[NV];
  double s0[ND], s1[ND];
  if (interior) {
    // The gating fields are first used ~400 instructions into the reaction and y at its very end;
    // under the 64-register cap ptxas sinks those loads next to their use (a second and third exposed
    // latency per warp).  Asking L1 for the lines now costs no register; the late loads then hit.
    // (Not for the 8 extra operand streams of K_RK4F: 4 blocks x 12 lines per thread overflow L1.)
    if (KIND != K_RK4F) {
      if (NV > 2) {   // only where the reaction is long enough to hide a DRAM latency (BOCF)
#pragma unroll
        for (int q = ND; q < NV; ++q) prefetch_l1(in + o + q * a.g.fstride);
      }
      if (KIND == K_BASE) {
#pragma unroll
        for (int q = 0; q < NV; ++q) prefetch_l1(yb + o + q * a.g.fstride);
      }
    }
#pragma unroll
    for (int q = 0; q < NV; ++q) zz[q] = ld2(in + o + q * a.g.fstride);
    // Stencil first: its neighbour loads go out together with the centre loads and are reduced to
    // two sums per diffusing field before the (register-hungry) reaction starts.  The RK operands
    // y / Y2 / Y3 are loaded after it, next to their use: with the kernel held to 64 registers
    // (32 warps per SM) the other warps cover that second latency, which measured faster
    // than keeping 12 more 128-bit loads in flight per thread (or prefetching them to L1).
#pragma unroll
    for (int q = 0; q < ND; ++q) {
      stencil_pair<STENCIL>(in + q * a.g.fstride + pz, row, x, pitch, zz[q], s0[q], s1[q]);
      if (D3) zarm_pair<STENCIL>(in + q * a.g.fstride, o, a.g.zstride, zz[q], s0[q], s1[q]);
    }
  } else {
    // rim blocks
    if (j >= ny || x >= nx) return;
    const int bc = a.g.boundary;
    if (x + 1 >= nx) {   // the last cell of an odd row: alone, boundary rule per neighbour
      const int oc = row + x;
      double z[NV], f[NV];
#pragma unroll
      for (int q = 0; q < NV; ++q) z[q] = in[o + q * a.g.fstride];
      MD::reaction(a.p, z, f);
#pragma unroll
      for (int q = 0; q < ND; ++q) {
        double s = stencil_edge<STENCIL>(in + q * a.g.fstride + pz, x, j, nx, ny, pitch, bc, z[q]);
        if (D3) s += zarm_edge<STENCIL>(in + q * a.g.fstride, oc, kz, a.g.nz, a.g.zstride, bc, z[q]);
        f[q] = fma(a.lapw[q], s, f[q]);
      }
      finish_cell<MD, KIND>(a, yb, Ab, Bb, ob, o, z, f);
      return;
    }
    // A pair inside the grid whose stencil may reach across the boundary keeps its 128-bit loads
    // (stencil_pair_bc, stage.cuh); in 3-D the z neighbours come from the reflected / wrapped plane.
#pragma unroll
    for (int q = 0; q < NV; ++q) zz[q] = ld2(in + o + q * a.g.fstride);
#pragma unroll
    for (int q = 0; q < ND; ++q) {
      const double2 c = zz[q];
      stencil_pair_bc<STENCIL>(in + q * a.g.fstride + pz, x, j, nx, ny, pitch, bc, c, s0[q], s1[q]);
      if (D3) {
        const double* V = in + q * a.g.fstride + row + x;
        const int nz = a.g.nz, zs = a.g.zstride;
        const double2 d1 = ld2(V + (long long)bidx(kz - 1, nz, bc) * zs), u1 = ld2(V + (long long)bidx(kz + 1, nz, bc) * zs);
        if (STENCIL == S_LAP9X4) {
          const double2 d2 = ld2(V + (long long)bidx(kz - 2, nz, bc) * zs), u2 = ld2(V + (long long)bidx(kz + 2, nz, bc) * zs);
          s0[q] += StencilZ<S_LAP9X4>::apply(c.x, d1.x, u1.x, d2.x, u2.x);
          s1[q] += StencilZ<S_LAP9X4>::apply(c.y, d1.y, u1.y, d2.y, u2.y);
        } else if (STENCIL == S_LAP5) {
          s0[q] += StencilZ<S_LAP5>::apply(c.x, d1.x, u1.x);
          s1[q] += StencilZ<S_LAP5>::apply(c.y, d1.y, u1.y);
        }
      }
    }
  }

  double z0[NV], z1[NV], f0[NV], f1[NV];
#pragma unroll
  for (int q = 0; q < NV; ++q) { z0[q] = zz[q].x; z1[q] = zz[q].y; }
  MD::reaction(a.p, z0, f0);
  MD::reaction(a.p, z1, f1);
#pragma unroll
  for (int q = 0; q < ND; ++q) {
    f0[q] = fma(a.lapw[q], s0[q], f0[q]);
    f1[q] = fma(a.lapw[q], s1[q], f1[q]);
  }
  if constexpr (KIND == K_RL || KIND == K_IE) {   // BOCF: u by Euler, the gates with frozen coefficients
    if constexpr (NV == 4) {
      double al0[3], be0[3], al1[3], be1[3];
      MD::gates(a.p, z0[0], al0, be0);
      MD::gates(a.p, z1[0], al1, be1);
      st2(ob + o, fma(a.dt, f0[0], z0[0]), fma(a.dt, f1[0], z1[0]));
#pragma unroll
      for (int g = 0; g < 3; ++g)
        st2(ob + o + (g + 1) * a.g.fstride, gate_step<KIND>(a.dt, z0[g + 1], al0[g], be0[g]),
            gate_step<KIND>(a.dt, z1[g + 1], al1[g], be1[g]));
    }
    return;
  }
#pragma unroll
  for (int q = 0; q < NV; ++q) {
    double2 yy = make_double2(0.0, 0.0), AA = yy, BB = yy;
    if (KIND != K_SELF) yy = ld2(yb + o + q * a.g.fstride);
    if (KIND == K_RK4F) { AA = ld2(Ab + o + q * a.g.fstride); BB = ld2(Bb + o + q * a.g.fstride); }
    double r0 = combine<KIND>(a.w_y, a.w_in, a.w_A, a.w_B, a.w_f, yy.x, z0[q], AA.x, BB.x, f0[q]);
    double r1 = combine<KIND>(a.w_y, a.w_in, a.w_A, a.w_B, a.w_f, yy.y, z1[q], AA.y, BB.y, f1[q]);
    st2(ob + o + q * a.g.fstride, r0, r1);
  }
}

template <class MD, int STENCIL, int KIND>
cudaError_t run(const Problem& pb, const StageLaunch& st, cudaStream_t stream) {
  StageArgs<MD> a;
  // unused operands alias the input so that every pointer the kernel forms is valid
  a.in = st.in; a.y = st.y ? st.y : st.in; a.A = st.A ? st.A : st.in; a.B = st.B ? st.B : st.in;
  a.out = st.out;
  a.g.nx = pb.nx; a.g.ny = pb.ny; a.g.pitch = pb.pitch; a.g.boundary = pb.boundary;
  a.g.nz = pb.nz; a.g.zstride = pb.zstride;
  a.g.fstride = pb.fstride; a.g.bstride = pb.bstride;
  a.w_y = st.w_y; a.w_in = st.w_in; a.w_A = st.w_A; a.w_B = st.w_B; a.w_f = st.w_f;
  a.dt = pb.dt;
  MD::derive(pb.params, a.p);
  for (int q = 0; q < MD::ND; ++q) a.lapw[q] = a.p.D[q] * stencil_norm(STENCIL) / (pb.dx * pb.dx);
  dim3 grid((pb.nx + 2 * TX - 1) / (2 * TX), (pb.ny + TY - 1) / TY, pb.batch * pb.nz), block(TX, TY);
  if (pb.nz > 1) {
    if constexpr (STENCIL == S_BOX9) return cudaErrorInvalidValue;   // no 3-D counterpart (rejected at create)
    else stage_kernel<MD, STENCIL, KIND, true><<<grid, block, 0, stream>>>(a);
  } else {
    stage_kernel<MD, STENCIL, KIND, false><<<grid, block, 0, stream>>>(a);
  }
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
  // one thread per output element of member blockIdx.y + 1
  const long long n = (long long)nx * ny * nv;
  const long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= n) return;
  const int i = (int)(e % nx);
  const long long rowf = e / nx;  // field * ny + j
  const long long src = rowf * pitch + i;
  const int b = blockIdx.y + 1;
  J[(long long)(b - 1) * n + e] = (Z[b * bstride + src] - Z[src]) / eps;
}

// rows [j0, j0 + nrows) of every field of every member <-> dense [batch * n_v][nrows][nx]
// (ghost-row exchange of a row-slab decomposition, include/cardiac.h cardiac_get_rows / _set_rows)
template <bool PACK>
__global__ void rows_kernel(double* __restrict__ Z, double* __restrict__ D, int nx, int nrows, int j0,
                            int pitch, long long fstride, long long n) {
  const long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= n) return;
  const int i = (int)(e % nx);
  const long long t = e / nx;
  const int j = (int)(t % nrows);
  const long long f = t / nrows;   // member * n_v + field
  const long long z = f * fstride + (long long)(j0 + j) * pitch + i;
  if (PACK) D[e] = Z[z];
  else Z[z] = D[e];
}

}  // namespace

cudaError_t launch_rows(const Problem& pb, double* state, int j0, int nrows, double* dense, bool pack,
                        cudaStream_t stream) {
  const long long n = (long long)pb.batch * pb.nv * nrows * pb.nx;
  if (n == 0) return cudaSuccess;
  const unsigned blocks = (unsigned)((n + 255) / 256);
  if (pack) rows_kernel<true><<<blocks, 256, 0, stream>>>(state, dense, pb.nx, nrows, j0, pb.pitch, pb.fstride, n);
  else rows_kernel<false><<<blocks, 256, 0, stream>>>(state, dense, pb.nx, nrows, j0, pb.pitch, pb.fstride, n);
  return cudaGetLastError();
}

cudaError_t launch_stage(const Problem& pb, const StageLaunch& st, cudaStream_t stream) {
  // DIRECT vs RING (bitwise identical results).  Measured on B200 (profiles/, r1 v4): with 32 warps
  // per SM the direct kernels hide their own load latency and win wherever a stage is bound by the
  // FP64 pipe or moves few bytes per cell; the TMA ring wins on the one stage that is purely
  // HBM-bound and operand-heavy — the last RK4 stage of the 4-field model (16 doubles in, 4 out per
  // cell; 6.3 TB/s = 96 % of the measured copy bandwidth, against 5.9 TB/s direct).
  // 3-D: the z-marching TMA ring (stream3d_kernels.cu) only where forced — measured slower than the direct
  // kernels at 256^3 for every model and stencil (8 - 16 warps per SM cannot hide its own shared-memory and FP64
  // latencies)
  if (pb.nz > 1 && pb.stage_impl == 2 && stage_ring3d_supported(pb, st.kind)) return launch_stage_ring3d(pb, st, stream);
  const long long cells = (long long)pb.nx * pb.ny * pb.batch;
  const bool ring_auto = st.kind == K_RK4F && pb.nv >= 4 && cells >= kRingMinCells;
  if (pb.stage_impl != 1 && (pb.stage_impl == 2 || ring_auto) && stage_ring_supported(pb, st.kind))
    return launch_stage_ring(pb, st, stream);
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
  const long long n = (long long)pb.nx * pb.ny * pb.nz * pb.nv;
  dim3 grid((unsigned)((n + 255) / 256), pb.batch - 1);
  jvp_kernel<<<grid, 256, 0, stream>>>(state, dst, pb.nx, pb.ny * pb.nz, pb.nv, pb.pitch, pb.bstride, eps);
  return cudaGetLastError();
}

}  // namespace cardiac
