// pairt_dispatch.cuh — host dispatch of plan PAIR / implementation TMA for one model; included by the
// per-model pairt_kernels_*.cu files so that the instantiations compile in parallel.
#pragma once
#include <atomic>

#include "pairt.cuh"

namespace cardiac {

// 64 x 24 tiles on 12 warps (two rows per warp, <= 168 registers).  Measured on B200, BOCF LAP9X4 RK4, us per
// step at 2048^2 / 4096^2: 248 / 963; 64 x 16 on 16 warps (128 registers) 256 / 1001; 64 x 20 on 20 warps
// (102 registers) 252 / 976 — more warps do not help: the schedulers' issue ports are what is busy
// (DESIGN.md "FP64 issue"), and the smaller tiles recompute a larger ring.
using PairTTile = PairTGeom<24, 384>;

template <class MD, int STENCIL, int KA, int KB, bool WRITE_P, class PG = PairTTile>
cudaError_t pairt_run(const Problem& pb, const PairTLaunch& pl, cudaStream_t stream) {
  using S = PairTShape<MD, STENCIL, KA, KB, PG>;
  auto kern = pair_tma_kernel<MD, STENCIL, KA, KB, WRITE_P, PG>;
  // per instantiation and device: the shared-memory limit and the size of the persistent grid (one CTA per SM)
  static PerDeviceOnce configured;
  static std::atomic<int> sms_of[64];
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 0 || dev >= 64) return cudaErrorInvalidDevice;
  e = configured.run([&] {
    cudaError_t e2 = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, S::SMEM_BYTES);
    if (e2 != cudaSuccess) return e2;
    int sms = 0;
    if ((e2 = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess) return e2;
    sms_of[dev].store(sms, std::memory_order_relaxed);
    return cudaSuccess;
  });
  if (e != cudaSuccess) return e;

  PairTArgs<MD> a;
  a.in = pl.in; a.y = pl.y ? pl.y : pl.in; a.out = pl.out; a.out2 = pl.out2 ? pl.out2 : pl.out;
  a.g.nx = pb.nx; a.g.ny = pb.ny; a.g.pitch = pb.pitch; a.g.boundary = pb.boundary;
  a.g.nz = 1; a.g.zstride = pb.zstride;
  a.g.fstride = pb.fstride; a.g.bstride = pb.bstride;
  a.a_wy = pl.a_wy; a.a_win = pl.a_win; a.a_wf = pl.a_wf;
  a.w_y = pl.w_y; a.w_in = pl.w_in; a.w_f = pl.w_f;
  a.p_wy = pl.p_wy; a.p_wA = pl.p_wA; a.p_wB = pl.p_wB;
  MD::derive(pb.params, a.p);
  for (int q = 0; q < MD::ND; ++q) a.lapw[q] = a.p.D[q] * stencil_norm(STENCIL) / (pb.dx * pb.dx);
  const long long tiles_x = (pb.nx + S::TW - 1) / S::TW, tiles_y = (pb.ny + S::TH - 1) / S::TH;
  const long long ntiles = tiles_x * tiles_y * pb.batch;
  if (ntiles >= (1LL << 31)) return cudaErrorInvalidValue;   // pair_tma_supported() said so
  a.tiles_x = (unsigned)tiles_x;
  a.ntiles = (unsigned)ntiles;
  a.per_member = make_fastdiv((unsigned)(tiles_x * tiles_y));
  a.per_row = make_fastdiv((unsigned)tiles_x);

  // tensor maps (cached by value): 4-D views (x, y, field, member) of the operand buffers
  CUtensorMap tm_inu, tm_ing, tm_yu, tm_yg, tm_p;
  if ((e = tensor_map_4d(a.in, pb, MD::ND, S::BW, S::BH, &tm_inu)) != cudaSuccess) return e;
  tm_ing = tm_yu = tm_yg = tm_p = tm_inu;
  if (S::NG > 0 && (e = tensor_map_4d(a.in + MD::ND * pb.fstride, pb, S::NG, S::WW, S::WH, &tm_ing)) != cudaSuccess)
    return e;
  if (KA == K_BASE) {
    if ((e = tensor_map_4d(a.y, pb, MD::ND, S::WW, S::WH, &tm_yu)) != cudaSuccess) return e;
    if (S::NG > 0 && (e = tensor_map_4d(a.y + MD::ND * pb.fstride, pb, S::NG, S::TW, S::TH, &tm_yg)) != cudaSuccess)
      return e;
  }
  if (S::HAS_P2) {
    if (!pl.P) return cudaErrorInvalidValue;
    if ((e = tensor_map_4d(pl.P, pb, MD::NV, S::TW, S::TH, &tm_p)) != cudaSuccess) return e;
  }
  long long grid = sms_of[dev].load(std::memory_order_relaxed);
  if (grid > ntiles) grid = ntiles;
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3((unsigned)grid);
  cfg.blockDim = dim3(S::NT);
  cfg.dynamicSmemBytes = S::SMEM_BYTES;
  cfg.stream = stream;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, kern, a, tm_inu, tm_ing, tm_yu, tm_yg, tm_p);
}

template <class MD, int STENCIL, class PG = PairTTile>
cudaError_t pairt_by_kind(const Problem& pb, const PairTLaunch& pl, cudaStream_t s) {
  if (pl.ka == K_SELF && pl.kb == K_BASE)
    return pl.out2 ? pairt_run<MD, STENCIL, K_SELF, K_BASE, true, PG>(pb, pl, s)     // RK4 substeps 1+2 (+ P)
                   : pairt_run<MD, STENCIL, K_SELF, K_BASE, false, PG>(pb, pl, s);   // Heun
  if (pl.ka == K_BASE && pl.kb == K_RK4F) return pairt_run<MD, STENCIL, K_BASE, K_RK4F, false, PG>(pb, pl, s);   // RK4 substeps 3+4
  if (pl.ka == K_SELF && pl.kb == K_SELF) return pairt_run<MD, STENCIL, K_SELF, K_SELF, false, PG>(pb, pl, s);   // two Euler steps
  return cudaErrorInvalidValue;
}

template <class MD>
cudaError_t pairt_by_stencil(const Problem& pb, const PairTLaunch& pl, cudaStream_t s) {
  switch (pb.stencil) {
    case S_LAP5: return pairt_by_kind<MD, S_LAP5>(pb, pl, s);
    case S_LAP9X4: return pairt_by_kind<MD, S_LAP9X4>(pb, pl, s);
    case S_BOX9: return pairt_by_kind<MD, S_BOX9>(pb, pl, s);
  }
  return cudaErrorInvalidValue;
}

}  // namespace cardiac
