// tilet.cuh — plan FUSED, implementation TMA: the on-chip tile engine of tile.cuh (all substeps of a time
// step, or four Euler steps, without leaving the SM) run by PERSISTENT CTAs whose windows arrive by TMA.
//
// Why: a fused_step_kernel CTA (one per SM, the whole register file) is a one-shot "load window -> wait ->
// n_s stages -> store"; nothing on the SM overlaps the load wait, the launch and the drain, and r1's cost
// model put that fixed part at the price of ~2000 cells per 3840-cell window.  Here one CTA per SM walks the
// tiles round-robin and the window of the NEXT tile is copied global -> shared by the TMA unit
// (cp.async.bulk.tensor, mbarrier complete_tx) while the stages of the current tile run.
//
//   buffers  three stage buffers [ND fields][SR rows][SP doubles] (tile.cuh layout: the box copy IS the padded
//            buffer, box = (EW + 2 PADX) x (EH + 2 R) from grid cell (x0 - H - PADX, y0 - H - R)) rotating
//            through the roles (input of this tile, ping-pong partner, input of the next tile), plus ONE
//            staging box [NG][EH][EW] for the non-diffusing fields, which are read into registers at the
//            start of a tile and whose box is re-filled for the next tile right after
//   stages   TileEngine::stage<S> unchanged: same instruction sequence per cell, same bits as plan FUSED
//   boundary the TMA unit zero-fills outside the grid; rim tiles overwrite the ghost cells within H = r n_s
//            of the grid with the cell the index reflects / wraps to (patch_box, pairt.cuh) before the
//            registers are loaded — the even extension of tile.cuh, valid where one reflection maps every
//            index (grids larger than window + halo; smaller grids stay with fused_step_kernel)
#pragma once
#include "pairt.cuh"   // patch_box
#include "tile.cuh"
#include "tma.cuh"

namespace cardiac {

template <class MD>
struct TileTArgs {
  TileArgs<MD> t;
  unsigned tiles_x, ntiles;
  FastDiv per_member, per_row;
};

template <class MD, int STENCIL, int INTEG, int KSTEPS, class TG>
struct TileTShape {
  using E = TileEngine<MD, STENCIL, INTEG, KSTEPS, TG>;
  static constexpr int NV = E::NV, ND = E::ND, NG = E::NG;
  static constexpr int BUF_BYTES = tma_align128(ND * E::FSZ * 8);
  static constexpr int GATE_BYTES = tma_align128((NG > 0 ? NG : 0) * TG::EW * TG::EH * 8);
  static constexpr unsigned TX_BUF = ND * E::FSZ * 8, TX_GATE = (NG > 0 ? NG : 0) * TG::EW * TG::EH * 8;
  static constexpr int OFF_GATE = 3 * BUF_BYTES, OFF_BAR = OFF_GATE + GATE_BYTES;
  static constexpr int SMEM_BYTES = OFF_BAR + 128;
  static_assert(SMEM_BYTES <= 227 * 1024, "three stage buffers of this window do not fit one SM");
  static_assert(E::NS == 2 || E::NS == 4, "the tile pipeline hangs its TMA requests on the barrier after substep 0");
};

template <class MD, int STENCIL, int INTEG, int KSTEPS, class TG>
__global__ void __launch_bounds__(TG::NT, TG::MINB)
    fused_tma_kernel(const __grid_constant__ TileTArgs<MD> ta, const __grid_constant__ CUtensorMap tm_u,
                     const __grid_constant__ CUtensorMap tm_g) {
  using E = TileEngine<MD, STENCIL, INTEG, KSTEPS, TG>;
  using S = TileTShape<MD, STENCIL, INTEG, KSTEPS, TG>;
  constexpr int NV = E::NV, ND = E::ND, NG = E::NG, R = E::R, H = E::H, PR = E::PR, NS = E::NS;
  constexpr int EW = E::EW, EH = E::EH, TW = E::TW, TH = E::TH, SP = E::SP, SR = E::SR, FSZ = E::FSZ, PADX = E::PADX;
  constexpr bool RK = E::RK;
  extern __shared__ __align__(1024) unsigned char tt_smem[];
  double* const gate = reinterpret_cast<double*>(tt_smem + S::OFF_GATE);   // [NG][EH][EW]
  uint64_t* const fullb = reinterpret_cast<uint64_t*>(tt_smem + S::OFF_BAR);   // one per stage buffer
  uint64_t* const fullg = fullb + 3;
  const TileArgs<MD>& a = ta.t;
  const int tid = threadIdx.x, tx = tid % TG::NTX, ty = tid / TG::NTX;
  auto buf = [&](int i) { return reinterpret_cast<double*>(tt_smem + i * S::BUF_BYTES); };

  auto issue_u = [&](unsigned t, int b) {
    const TilePos tp = tile_pos_of(t, ta.per_member, ta.per_row, ta.tiles_x, TW, TH);
    mbar_arrive_expect_tx(fullb + b, S::TX_BUF);
    tma_load_4d(buf(b), &tm_u, tp.x0 - H - PADX, tp.y0 - H - R, 0, tp.bz, fullb + b);
  };
  auto issue_g = [&](unsigned t) {
    const TilePos tp = tile_pos_of(t, ta.per_member, ta.per_row, ta.tiles_x, TW, TH);
    mbar_arrive_expect_tx(fullg, S::TX_GATE);
    tma_load_4d(gate, &tm_g, tp.x0 - H, tp.y0 - H, 0, tp.bz, fullg);
  };

  if (tid == 0) {
#pragma unroll
    for (int i = 0; i < 4; ++i) mbar_init(fullb + i, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  }
  __syncthreads();
  asm volatile("griddepcontrol.wait;" ::: "memory");
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  if (tid == 0 && blockIdx.x < ta.ntiles) {
    issue_u(blockIdx.x, 0);
    if (NG > 0) issue_g(blockIdx.x);
  }

  int in = 0, partner = 1, pre = 2;      // roles of the three stage buffers
  unsigned phb = 0, phg = 0;             // parity of the next completion of each barrier (bit i: buffer i)
  for (unsigned t = blockIdx.x; t < ta.ntiles; t += gridDim.x) {
    const TilePos tp = tile_pos_of(t, ta.per_member, ta.per_row, ta.tiles_x, TW, TH);
    const int bx = tp.x0 / TW, by = tp.y0 / TH;
    const long long base = (long long)tp.bz * a.g.bstride;
    const unsigned long long tn = (unsigned long long)t + gridDim.x;   // the next tile of this CTA
    double* const cur0 = buf(in);
    mbar_wait(fullb + in, (phb >> in) & 1u);
    phb ^= 1u << in;
    if (NG > 0) { mbar_wait(fullg, phg); phg ^= 1; }
    const int wx0 = tp.x0 - H, wy0 = tp.y0 - H;   // grid cell of window cell (0, 0)
    if (wx0 < 0 || wx0 + EW > a.g.nx || wy0 < 0 || wy0 + EH > a.g.ny) {   // rim tile: even / periodic extension
      patch_box<H>(cur0, ND, SP, SR, wx0 - PADX, wy0 - R, a.in + base, a.g, tid, TG::NT);
      if (NG > 0) patch_box<H>(gate, NG, EW, EH, wx0, wy0, a.in + base + ND * a.g.fstride, a.g, tid, TG::NT);
      asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
      __syncthreads();
    }
    // registers of the 2 x PR patch: y (RK schemes) and the non-diffusing fields
    typename E::Patch st;
    {
      const double* s0 = cur0 + (R + PR * ty) * SP + PADX + 2 * tx;
#pragma unroll
      for (int k = 0; k < PR; ++k) {
#pragma unroll
        for (int q = 0; q < NV; ++q) {
          double2 v;
          if (q < ND) v = *reinterpret_cast<const double2*>(s0 + q * FSZ + k * SP);
          else v = *reinterpret_cast<const double2*>(gate + (q - ND) * EW * EH + (PR * ty + k) * EW + 2 * tx);
          if (q >= ND) { st.g[k][0][q >= ND ? q - ND : 0] = v.x; st.g[k][1][q >= ND ? q - ND : 0] = v.y; }
          if (RK) { st.y[k][0][q] = v.x; st.y[k][1][q] = v.y; }
        }
      }
    }

    // the substeps: in -> partner -> in -> ... ; the last one writes global memory
    double* out = a.out + base;
    double* c = cur0;
    double* n = buf(partner);
    {
      E::template stage<0>(a, out, bx, by, tx, ty, c, n, st);
      // One barrier does three jobs.  (i) Substep 0 is complete.  (ii) Every thread has finished the LAST substep of
      // the previous tile, which read that tile's partner buffer = this tile's `pre`: the next tile's window may
      // land there (its generic-proxy stores are fenced against the async-proxy write first).  (iii) Every thread
      // has read the staging box of the non-diffusing fields: the next tile's may land.  No barrier is needed at
      // the END of a tile: substep 0 of the next tile writes the buffer that was this tile's input, last read in the
      // second-to-last substep, which the barrier before the last substep already closed.
      asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
      __syncthreads();
      if (tid == 0 && tn < ta.ntiles) {
        issue_u((unsigned)tn, pre);
        if (NG > 0) issue_g((unsigned)tn);
      }
      E::template stage<1>(a, out, bx, by, tx, ty, n, c, st);
      if constexpr (NS == 4) {
        __syncthreads();
        E::template stage<2>(a, out, bx, by, tx, ty, c, n, st);
        __syncthreads();
        E::template stage<3>(a, out, bx, by, tx, ty, n, c, st);
      }
    }
    const int o = in; in = pre; pre = partner; partner = o;   // (in, partner, pre) <- (pre, in, partner)
  }
}

}  // namespace cardiac
