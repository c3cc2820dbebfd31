// pair_dispatch.cuh — host dispatch of plan PAIR for one model; included by the per-model
// pair_kernels_*.cu files so that the instantiations compile in parallel.
#pragma once
#include "pair.cuh"

namespace cardiac {

// Tile: 64 x 24 cells, 256 threads (a thread keeps its column pair and walks 3 rows), TWO CTAs per SM at
// 128 registers: the interior path requests every global operand of a row before the reaction starts
// (one exposed memory latency per row instead of three), which needs the registers.  Shared memory per
// CTA = 8 B x (n_d x 68 x (24+2r) + (n_v-n_d) x 64 x 24): 52 KB for BOCF with r = 2.  Measured on B200,
// 2048^2 / 4096^2 BOCF LAP9X4 RK4, us per step: 310 / 1054; without the early loads 341 / 1188; three
// CTAs at 80 registers 335 / 1126; four at 64 registers (spills in the row loops) 415 / 1365; register
// double-buffering of the next row's stencil inputs 319 / 1115 (not kept).
using PairTile = PairGeom<64, 24, 256, 2>;

template <class MD, int STENCIL, int KA, int KB, bool STORE_MID>
cudaError_t pair_run(const Problem& pb, const PairLaunch& pl, cudaStream_t stream) {
  using PG = PairTile;
  using S = PairShape<MD, STENCIL, PG>;
  auto kern = pair_kernel<MD, STENCIL, KA, KB, STORE_MID, PG>;
  static PerDeviceOnce configured;  // per instantiation and device
  cudaError_t ec = configured.run(
      [&] { return cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, S::SMEM_BYTES); });
  if (ec != cudaSuccess) return ec;
  if (KB == K_RK4F && pl.B != pl.in) return cudaErrorInvalidValue;   // Y3 is read as substep A's input
  PairArgs<MD> a;
  // unused operands alias valid buffers so that every pointer the kernel forms is valid
  a.in = pl.in; a.y = pl.y ? pl.y : pl.in; a.A = pl.A ? pl.A : pl.in; a.B = pl.B ? pl.B : pl.in;
  a.mid = pl.mid ? pl.mid : pl.out; a.out = pl.out;
  a.g.nx = pb.nx; a.g.ny = pb.ny; a.g.pitch = pb.pitch; a.g.boundary = pb.boundary;
  a.g.nz = 1; a.g.zstride = pb.zstride;
  a.g.fstride = pb.fstride; a.g.bstride = pb.bstride;
  a.a_wy = pl.a_wy; a.a_win = pl.a_win; a.a_wf = pl.a_wf;
  a.w_y = pl.w_y; a.w_in = pl.w_in; a.w_A = pl.w_A; a.w_B = pl.w_B; a.w_f = pl.w_f;
  MD::derive(pb.params, a.p);
  for (int q = 0; q < MD::ND; ++q) a.lapw[q] = a.p.D[q] * stencil_norm(STENCIL) / (pb.dx * pb.dx);
  dim3 grid((pb.nx + PG::TW - 1) / PG::TW, (pb.ny + PG::TH - 1) / PG::TH, pb.batch);
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = grid;
  cfg.blockDim = dim3(PG::NT);
  cfg.dynamicSmemBytes = S::SMEM_BYTES;
  cfg.stream = stream;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, kern, a);
}

template <class MD, int STENCIL>
cudaError_t pair_by_kind(const Problem& pb, const PairLaunch& pl, cudaStream_t s) {
  if (pl.ka == K_SELF && pl.kb == K_BASE)
    return pl.mid ? pair_run<MD, STENCIL, K_SELF, K_BASE, true>(pb, pl, s)     // RK4 substeps 1+2
                  : pair_run<MD, STENCIL, K_SELF, K_BASE, false>(pb, pl, s);   // Heun
  if (pl.ka == K_BASE && pl.kb == K_RK4F && !pl.mid)
    return pair_run<MD, STENCIL, K_BASE, K_RK4F, false>(pb, pl, s);            // RK4 substeps 3+4
  if (pl.ka == K_SELF && pl.kb == K_SELF && !pl.mid)
    return pair_run<MD, STENCIL, K_SELF, K_SELF, false>(pb, pl, s);            // two Euler steps
  return cudaErrorInvalidValue;
}

template <class MD>
cudaError_t pair_by_stencil(const Problem& pb, const PairLaunch& pl, cudaStream_t s) {
  switch (pb.stencil) {
    case S_LAP5: return pair_by_kind<MD, S_LAP5>(pb, pl, s);
    case S_LAP9X4: return pair_by_kind<MD, S_LAP9X4>(pb, pl, s);
    case S_BOX9: return pair_by_kind<MD, S_BOX9>(pb, pl, s);
  }
  return cudaErrorInvalidValue;
}

}  // namespace cardiac
