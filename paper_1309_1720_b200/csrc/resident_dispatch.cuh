// resident_dispatch.cuh — host dispatch of plan PERSISTENT for one model; included by the per-model
// resident_kernels_*.cu files so that the instantiations compile in parallel.
#pragma once
#include "plans.h"
#include "resident.cuh"

namespace cardiac {

// pairs per thread: 4 (4096 cells per CTA) for the two-field models; the 4-field model keeps 11
// doubles per cell in registers, so 2 (2048 cells)
template <class MD>
struct ResidentPairs {
  static constexpr int KP = MD::NV > 2 ? 2 : 4;
};

template <class MD, int STENCIL, int INTEG, int CPT, int KP = ResidentPairs<MD>::KP>
cudaError_t resident_run(const Problem& pb, const ResidentLaunch& rl, cudaStream_t stream) {
  constexpr int R = stencil_radius(STENCIL);
  auto kern = resident_kernel<MD, STENCIL, INTEG, KP, CPT>;
  ResidentArgs<MD> a;
  a.in = rl.state; a.out = rl.state;
  a.g.nx = pb.nx; a.g.ny = pb.ny; a.g.pitch = pb.pitch; a.g.boundary = pb.boundary;
  a.g.nz = 1; a.g.zstride = pb.zstride;
  a.g.fstride = pb.fstride; a.g.bstride = pb.bstride;
  a.nsteps = rl.nsteps;
  const ResidentShape rs = resident_shape(pb);
  if (rs.csize == 0) return cudaErrorInvalidValue;
  a.npx = (pb.nx + 1) / 2;
  a.slab = rs.slab;
  a.csize = rs.csize;
  a.sp = 2 * a.npx + 4;
  a.sr = rs.slab + 2 * R;
  const double dt = pb.dt;
  for (int s = 0; s < 4; ++s) a.a_dt[s] = a.b_dt[s] = 0.0;
  if (INTEG == I_RK4) {
    a.a_dt[0] = 0.5 * dt; a.a_dt[1] = 0.5 * dt; a.a_dt[2] = dt;
    a.b_dt[0] = dt / 6.0; a.b_dt[1] = dt / 3.0; a.b_dt[2] = dt / 3.0; a.b_dt[3] = dt / 6.0;
  } else if (INTEG == I_HEUN) {
    a.a_dt[0] = dt; a.b_dt[0] = 0.5 * dt; a.b_dt[1] = 0.5 * dt;
  } else {
    a.a_dt[0] = dt;
  }
  MD::derive(pb.params, a.p);
  for (int q = 0; q < MD::ND; ++q) a.lapw[q] = a.p.D[q] * stencil_norm(STENCIL) / (pb.dx * pb.dx);
  const size_t smem = rs.smem;
  if ((long long)a.npx * rs.slab * (3 - CPT) > (long long)kResidentThreads * KP) return cudaErrorInvalidValue;
  // per instantiation and device: clusters of 16 CTAs, and the largest slab resident_shape() ever asks for
  static PerDeviceOnce configured;
  cudaError_t ec = configured.run([&] {
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
    if (e != cudaSuccess) return e;
    return cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kResidentMaxSmem);
  });
  if (ec != cudaSuccess) return ec;
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3((unsigned)pb.batch * rs.csize);
  cfg.blockDim = dim3(kResidentThreads);
  cfg.dynamicSmemBytes = smem;
  cfg.stream = stream;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeClusterDimension;
  attr[0].val.clusterDim.x = rs.csize;
  attr[0].val.clusterDim.y = 1;
  attr[0].val.clusterDim.z = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, kern, a);
}

template <class MD, int STENCIL>
cudaError_t resident_by_integrator(const Problem& pb, const ResidentLaunch& rl, cudaStream_t s) {
  // one cell per thread and unit where the slab leaves the threads the room (resident.cuh, CPT)
  const ResidentShape rs = resident_shape(pb);
  // FHN only while every thread has at most one unit: a thread's units run one after the other, and two
  // light cells cost more than one pair (Euler 96^2: 1.24 us per step as cells, 0.95 as pairs); Karma and
  // BOCF wherever the cells fit (Karma RK4 96^2: 5.9 against 6.9 us, BOCF RK4 80^2: 8.5 against 10.8 us)
  const long long ncell = 2LL * ((pb.nx + 1) / 2) * rs.slab;
  const bool cells = ncell <= (long long)kResidentThreads * (MD::NV > 2 || pb.model != 0 ? ResidentPairs<MD>::KP : 1);
  // the smallest grids (at most one cell per thread: cfg 1) run an instantiation without the loop over units: a
  // substep there is the latency of ONE warp's instruction sequence, and the unit loop is part of it
  if (cells && ncell <= kResidentThreads) {
    switch (pb.integrator) {
      case I_EULER: return resident_run<MD, STENCIL, I_EULER, 1, 1>(pb, rl, s);
      case I_HEUN: return resident_run<MD, STENCIL, I_HEUN, 1, 1>(pb, rl, s);
      case I_RK4: return resident_run<MD, STENCIL, I_RK4, 1, 1>(pb, rl, s);
    }
  }
  switch (pb.integrator) {
    case I_EULER: return cells ? resident_run<MD, STENCIL, I_EULER, 1>(pb, rl, s) : resident_run<MD, STENCIL, I_EULER, 2>(pb, rl, s);
    case I_HEUN: return cells ? resident_run<MD, STENCIL, I_HEUN, 1>(pb, rl, s) : resident_run<MD, STENCIL, I_HEUN, 2>(pb, rl, s);
    case I_RK4: return cells ? resident_run<MD, STENCIL, I_RK4, 1>(pb, rl, s) : resident_run<MD, STENCIL, I_RK4, 2>(pb, rl, s);
  }
  return cudaErrorInvalidValue;
}

template <class MD>
cudaError_t resident_by_stencil(const Problem& pb, const ResidentLaunch& rl, cudaStream_t s) {
  switch (pb.stencil) {
    case S_LAP5: return resident_by_integrator<MD, S_LAP5>(pb, rl, s);
    case S_LAP9X4: return resident_by_integrator<MD, S_LAP9X4>(pb, rl, s);
    case S_BOX9: return resident_by_integrator<MD, S_BOX9>(pb, rl, s);
  }
  return cudaErrorInvalidValue;
}

}  // namespace cardiac
