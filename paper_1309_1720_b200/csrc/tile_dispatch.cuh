// tile_dispatch.cuh — kernels and host dispatch of plan FUSED for one model; included by the
// per-model tile_kernels_*.cu files so that the (large, fully unrolled) instantiations compile in
// parallel.
#pragma once
#include "plans.h"
#include "tile.cuh"

namespace cardiac {

// window geometry per (model, halo): 2*NTX x PR*NTY cells, NTX*NTY threads, one CTA per SM.
// The 4-field ionic model keeps 11 doubles per cell in registers, so its patches are smaller.
template <class MD, int H, int WIN>
struct FusedGeom {
  using type = TileGeom<40, 12, 4>;  // 80 x 48 window, 480 threads
};
// Mid-size grids (the paper's own range, 256^2 - 768^2) give the large window fewer
// tiles than there are SMs, and a step then costs one CTA lifetime (~7.5 us) whatever the size: the
// small window halves the cells per thread (2 x 2 instead of 2 x 4) and lets two CTAs share an SM.
template <class MD, int H>
struct FusedGeom<MD, H, 2> {
  using type = TileGeom<24, 20, 2, 2>;  // 48 x 40 window, 480 threads, 2 CTAs per SM
};
// With a halo of 8 a step costs (waves of CTAs) x (window area): 64 x 56 cells (tile 48 x 40, 448 threads)
// is 7 % less area than 80 x 48 (tile 64 x 32) and tiles 512^2 with 143 CTAs — still one wave of the 148 SMs.
template <class MD, int H>
struct FusedGeom<MD, H, 3> {
  using type = TileGeom<32, 14, 4>;
};
// two more one-CTA-per-SM windows for grids that the others tile into a badly filled last wave
template <class MD, int H>
struct FusedGeom<MD, H, 4> {
  using type = TileGeom<32, 12, 4>;  // 64 x 48 window, 384 threads
};
template <class MD, int H>
struct FusedGeom<MD, H, 5> {
  using type = TileGeom<28, 12, 4>;  // 56 x 48 window, 336 threads
};
// the 64 x 56 window again with HALF the cells per thread (2 x 2) and twice the threads (64 registers): 28 warps
// on the SM.  Measured on B200 (RK4): worse for FHN LAP9X4 (spills; 31 against 39 Gcell-step/s), better for
// Karma LAP5, whose stage is bound by instruction issue: 1024^2 41 against 38.5 with one CTA per tile, and
// 42 / 47 / 49.5 at 1024^2 / 2048^2 / 4096^2 with the TMA-fed persistent CTAs (tilet.cuh) against 38 / 40 / 41.
template <class MD, int H>
struct FusedGeom<MD, H, 7> {
  using type = TileGeom<32, 28, 2>;  // 64 x 56 window, 896 threads
};
// Small grids (one wave of tiles) pay one CTA lifetime per time step, and the lifetime grows with the rows a thread
// walks per substep: a 64 x 32 window on 1024 threads x ONE row of a pair each.  Measured (RK4, us per step, against
// the windows above): FHN LAP9X4 256^2 5.2 / 6.1, 320^2 5.1 / 6.3; Karma LAP5 256^2 5.7 / 6.3, 384^2 6.1 / 6.4; FHN LAP5
// (halo 4) loses to the 48 x 40 window (4.8 / 4.35).  Two waves always lose.
template <class MD, int H>
struct FusedGeom<MD, H, 8> {
  using type = TileGeom<32, 32, 1>;  // 64 x 32 window, 1024 threads
};
template <int VARIANT, int H, int WIN>
struct FusedGeom<Model<M_BOCF, VARIANT>, H, WIN> {
  using type = TileGeom<24, 16, 2>;  // 48 x 32 window, 384 threads
};

template <class MD, int STENCIL, int INTEG, int KSTEPS, class TG>
__global__ void __launch_bounds__(TG::NT, TG::MINB)
    fused_step_kernel(const __grid_constant__ TileArgs<MD> a) {
  using E = TileEngine<MD, STENCIL, INTEG, KSTEPS, TG>;
  extern __shared__ double2 smem_fused[];
  // programmatic dependent launch: this grid may be scheduled while the previous time step's grid
  // drains; every global access below waits for that grid to complete and flush
  asm volatile("griddepcontrol.wait;" ::: "memory");
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  const long long base = (long long)blockIdx.z * a.g.bstride;
  E::run(a, a.in + base, a.out + base, blockIdx.x, blockIdx.y, reinterpret_cast<double*>(smem_fused));
}

template <class MD>
void fill_tile_args(const Problem& pb, int stencil, TileArgs<MD>& a) {
  a.g.nx = pb.nx; a.g.ny = pb.ny; a.g.pitch = pb.pitch; a.g.boundary = pb.boundary;
  a.g.nz = 1; a.g.zstride = pb.zstride;
  a.g.fstride = pb.fstride; a.g.bstride = pb.bstride;
  const double dt = pb.dt;
  for (int s = 0; s < 4; ++s) a.a_dt[s] = a.b_dt[s] = 0.0;
  if (pb.integrator == I_RK4) {
    // Y2 = y + dt/2 k1, Y3 = y + dt/2 k2, Y4 = y + dt k3; y+ = y + dt/6 (k1 + 2 k2 + 2 k3 + k4)
    a.a_dt[0] = 0.5 * dt; a.a_dt[1] = 0.5 * dt; a.a_dt[2] = dt;
    a.b_dt[0] = dt / 6.0; a.b_dt[1] = dt / 3.0; a.b_dt[2] = dt / 3.0; a.b_dt[3] = dt / 6.0;
  } else if (pb.integrator == I_HEUN) {
    a.a_dt[0] = dt; a.b_dt[0] = 0.5 * dt; a.b_dt[1] = 0.5 * dt;
  } else {
    a.a_dt[0] = dt;
  }
  MD::derive(pb.params, a.p);
  for (int q = 0; q < MD::ND; ++q) a.lapw[q] = a.p.D[q] * stencil_norm(stencil) / (pb.dx * pb.dx);
}

template <class MD, int STENCIL, int INTEG, int KSTEPS, int WIN = 1>
cudaError_t fused_run(const Problem& pb, const TileLaunch& tl, cudaStream_t stream) {
  constexpr int H = stencil_radius(STENCIL) * StepScheme<INTEG, KSTEPS>::NS;
  using TG = typename FusedGeom<MD, H, WIN>::type;
  using E = TileEngine<MD, STENCIL, INTEG, KSTEPS, TG>;
  auto kern = fused_step_kernel<MD, STENCIL, INTEG, KSTEPS, TG>;
  static PerDeviceOnce configured;  // per instantiation and device
  cudaError_t ec = configured.run(
      [&] { return cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, E::SMEM_BYTES); });
  if (ec != cudaSuccess) return ec;
  TileArgs<MD> a;
  fill_tile_args<MD>(pb, STENCIL, a);
  a.in = tl.in; a.out = tl.out;
  dim3 grid((pb.nx + E::TW - 1) / E::TW, (pb.ny + E::TH - 1) / E::TH, pb.batch);
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = grid;
  cfg.blockDim = dim3(TG::NT);
  cfg.dynamicSmemBytes = E::SMEM_BYTES;
  cfg.stream = stream;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, kern, a);
}

template <class MD, int STENCIL>
cudaError_t fused_by_integrator(const Problem& pb, const TileLaunch& tl, cudaStream_t s) {
  switch (pb.integrator) {
    case I_RK4:
      if constexpr (MD::NV <= 2) {
        if (tl.window == 2) return fused_run<MD, STENCIL, I_RK4, 1, 2>(pb, tl, s);
        if (tl.window == 3) return fused_run<MD, STENCIL, I_RK4, 1, 3>(pb, tl, s);
        if (tl.window == 4) return fused_run<MD, STENCIL, I_RK4, 1, 4>(pb, tl, s);
        if (tl.window == 5) return fused_run<MD, STENCIL, I_RK4, 1, 5>(pb, tl, s);
        if (tl.window == 7) return fused_run<MD, STENCIL, I_RK4, 1, 7>(pb, tl, s);
        if (tl.window == 8) return fused_run<MD, STENCIL, I_RK4, 1, 8>(pb, tl, s);
      }
      return fused_run<MD, STENCIL, I_RK4, 1>(pb, tl, s);
    case I_HEUN:
      if constexpr (MD::NV <= 2)
        if (tl.window == 2) return fused_run<MD, STENCIL, I_HEUN, 1, 2>(pb, tl, s);
      return fused_run<MD, STENCIL, I_HEUN, 1>(pb, tl, s);
    case I_EULER:
      if (tl.ksteps == 1) return fused_run<MD, STENCIL, I_EULER, 1>(pb, tl, s);
      if (tl.ksteps == kEulerBlock) return fused_run<MD, STENCIL, I_EULER, kEulerBlock>(pb, tl, s);
      break;
  }
  return cudaErrorInvalidValue;
}

template <class MD>
cudaError_t fused_by_stencil(const Problem& pb, const TileLaunch& tl, cudaStream_t s) {
  switch (pb.stencil) {
    case S_LAP5: return fused_by_integrator<MD, S_LAP5>(pb, tl, s);
    case S_LAP9X4: return fused_by_integrator<MD, S_LAP9X4>(pb, tl, s);
    case S_BOX9: return fused_by_integrator<MD, S_BOX9>(pb, tl, s);
  }
  return cudaErrorInvalidValue;
}

}  // namespace cardiac
