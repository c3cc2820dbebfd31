// tilet_dispatch.cuh — host dispatch of plan FUSED / implementation TMA for one model; included by the
// per-model tilet_kernels_*.cu files.
#pragma once
#include <atomic>

#include "tile_dispatch.cuh"
#include "tilet.cuh"

namespace cardiac {

template <class MD, int STENCIL, int INTEG, int KSTEPS, int WIN = 1>
cudaError_t fusedt_run(const Problem& pb, const TileLaunch& tl, cudaStream_t stream) {
  constexpr int H = stencil_radius(STENCIL) * StepScheme<INTEG, KSTEPS>::NS;
  using TG = typename FusedGeom<MD, H, WIN>::type;
  using E = TileEngine<MD, STENCIL, INTEG, KSTEPS, TG>;
  using S = TileTShape<MD, STENCIL, INTEG, KSTEPS, TG>;
  auto kern = fused_tma_kernel<MD, STENCIL, INTEG, KSTEPS, TG>;
  // one reflection / wrap must map every window index (tile.cuh `once_x`): smaller grids keep fused_step_kernel
  if (pb.nx <= H + E::TW || pb.ny <= H + E::TH) return cudaErrorInvalidValue;
  static PerDeviceOnce configured;   // per instantiation and device
  static std::atomic<int> grid_of[64];
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 0 || dev >= 64) return cudaErrorInvalidDevice;
  e = configured.run([&] {
    cudaError_t e2 = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, S::SMEM_BYTES);
    if (e2 != cudaSuccess) return e2;
    int sms = 0, occ = 0;
    if ((e2 = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess) return e2;
    if ((e2 = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, TG::NT, S::SMEM_BYTES)) != cudaSuccess) return e2;
    if (occ < 1) return cudaErrorLaunchOutOfResources;
    grid_of[dev].store(sms * occ, std::memory_order_relaxed);
    return cudaSuccess;
  });
  if (e != cudaSuccess) return e;

  TileTArgs<MD> ta;
  fill_tile_args<MD>(pb, STENCIL, ta.t);
  ta.t.in = tl.in; ta.t.out = tl.out;
  const long long tiles_x = (pb.nx + E::TW - 1) / E::TW, tiles_y = (pb.ny + E::TH - 1) / E::TH;
  const long long ntiles = tiles_x * tiles_y * pb.batch;
  if (ntiles >= (1LL << 31)) return cudaErrorInvalidValue;
  ta.tiles_x = (unsigned)tiles_x;
  ta.ntiles = (unsigned)ntiles;
  ta.per_member = make_fastdiv((unsigned)(tiles_x * tiles_y));
  ta.per_row = make_fastdiv((unsigned)tiles_x);
  CUtensorMap tm_u, tm_g;
  if ((e = tensor_map_4d(tl.in, pb, MD::ND, E::SP, E::SR, &tm_u)) != cudaSuccess) return e;
  tm_g = tm_u;
  if (E::NG > 0 && (e = tensor_map_4d(tl.in + MD::ND * pb.fstride, pb, E::NG, TG::EW, TG::EH, &tm_g)) != cudaSuccess) return e;
  long long grid = grid_of[dev].load(std::memory_order_relaxed);
  if (grid > ntiles) grid = ntiles;
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3((unsigned)grid);
  cfg.blockDim = dim3(TG::NT);
  cfg.dynamicSmemBytes = S::SMEM_BYTES;
  cfg.stream = stream;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, kern, ta, tm_u, tm_g);
}

// the windows of the two-field models (tile_dispatch.cuh); the 4-field model runs plan PAIR instead
template <class MD, int STENCIL>
cudaError_t fusedt_by_integrator(const Problem& pb, const TileLaunch& tl, cudaStream_t s) {
  switch (pb.integrator) {
    case I_RK4:
      if (tl.window == 2) return fusedt_run<MD, STENCIL, I_RK4, 1, 2>(pb, tl, s);
      if (tl.window == 3) return fusedt_run<MD, STENCIL, I_RK4, 1, 3>(pb, tl, s);
      if (tl.window == 7) return fusedt_run<MD, STENCIL, I_RK4, 1, 7>(pb, tl, s);
      return fusedt_run<MD, STENCIL, I_RK4, 1>(pb, tl, s);
    case I_HEUN:
      if (tl.window == 2) return fusedt_run<MD, STENCIL, I_HEUN, 1, 2>(pb, tl, s);
      return fusedt_run<MD, STENCIL, I_HEUN, 1>(pb, tl, s);
    case I_EULER:
      if (tl.ksteps == kEulerBlock) return fusedt_run<MD, STENCIL, I_EULER, kEulerBlock>(pb, tl, s);
      break;
  }
  return cudaErrorInvalidValue;
}

template <class MD>
cudaError_t fusedt_by_stencil(const Problem& pb, const TileLaunch& tl, cudaStream_t s) {
  switch (pb.stencil) {
    case S_LAP5: return fusedt_by_integrator<MD, S_LAP5>(pb, tl, s);
    case S_LAP9X4: return fusedt_by_integrator<MD, S_LAP9X4>(pb, tl, s);
    case S_BOX9: return fusedt_by_integrator<MD, S_BOX9>(pb, tl, s);
  }
  return cudaErrorInvalidValue;
}

}  // namespace cardiac
