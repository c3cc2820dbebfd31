// pairt.cuh — plan PAIR, implementation TMA: two consecutive RK substeps per launch (pair.cuh), with every
// global operand moved into shared memory by the TMA unit AHEAD of the warps that consume it.
//
// Why (ncu, profiles/r2_v0_cfg4_pair_*): the direct PAIR kernels are bound by neither HBM (2.5-3.1 TB/s)
// nor the FP64 pipe (58-63 % active); their time is, to a few per cent, the SUM of the two — a warp loads,
// waits an L2 latency, computes ~650 instructions, and with 4 warps per scheduler at 128 registers nothing
// overlaps the wait (long scoreboard 18 % / 29 % of all stall samples, barrier 5 %).  Here the warps never
// touch global memory for input: persistent CTAs (one per SM) walk the tiles round-robin; one elected
// thread issues the box copies (cp.async.bulk.tensor, mbarrier complete_tx) of the NEXT tile's operands
// while the 12 warps compute the current one from shared memory.
//
//   tile     64 x 24 cells of one batch member; 384 threads = 12 warps, a warp = 2 tile rows, a lane = an
//            x-adjacent pair of cells (128-bit shared-memory accesses)
//   phase 1  substep A on the tile plus a ring of r cells (ring: the diffusing fields only) from the P1 slot:
//            [in: diffusing fields, box 72 x (24+4r)] [in: gating fields on the window 68 x (24+2r)]
//            and, when substep A is K_BASE, [y: diffusing on the window] [y: gating on the tile];
//            result -> shared window (as in pair.cuh)
//   phase 2  substep B on the tile from the window; its pointwise operand comes from the P1 slot (y = `in`
//            when substep A is K_SELF) or from the P2 slot [P on the tile, all fields]; result -> global
//   overlap  substep A = K_SELF (RK4 launch 1, Heun, Euler x 2): two P1 slots, the tile after next is
//            requested when a tile is done.  Substep A = K_BASE (RK4 launch 2): one P1 and one P2 slot;
//            P1 of the next tile is requested after phase 1 (in flight during phase 2), P2 after phase 2
//            (in flight during the next phase 1).
//
// RK4, accumulator-free, same combinations and weights as plan STAGE (hence the same bits):
//   launch 1:  Y2 = y + dt/2 f(y) [shared],  Y3 = y + dt/2 f(Y2) -> global,
//              P = (2 Y3 + Y2 - y)/3 -> global   (everything of y+ that does not depend on Y4; phase 2
//              holds y, Y2 and Y3 at that point, so Y2 itself never reaches memory)
//   launch 2:  Y4 = y + dt f(Y3) [shared],   y+ = P + Y4/3 + dt/6 f(Y4) -> global (may overwrite P)
// 4 + 8 and 12 + 4 doubles per cell and field, as the direct implementation.
//
// Boundary (PAPER.md:104 Fig. 1, :114): the TMA unit zero-fills what lies outside the grid.  On rim tiles
// the ghost cells within 2r (input boxes) / r (window boxes) of the grid are overwritten with the cell the
// index reflects or wraps to before phase 1 runs; a ghost window cell evaluated from such an evenly
// extended input reproduces its image bitwise (the stencils are sums of west+east / south+north pairs), so
// neither phase has boundary logic.
#pragma once
#include "plans.h"
#include "stage.cuh"
#include "tma.cuh"

namespace cardiac {

template <class MD>
struct PairTArgs {
  const double* in;   // input of substep A (the rim patch reads it directly)
  const double* y;    // state at the start of the time step (substep A = K_BASE: rim patch)
  double* out;        // result of substep B
  double* out2;       // WRITE_P: where P goes
  Geom g;
  double a_wy, a_win, a_wf;           // substep A
  double w_y, w_in, w_f;              // substep B (K_RK4F: w_in, w_f and the P read back)
  double p_wy, p_wA, p_wB;            // WRITE_P: P = p_wB Y3 + (p_wA Y2 + p_wy y)
  double lapw[MD::ND];
  typename MD::Params p;
  unsigned tiles_x, ntiles;
  FastDiv per_member, per_row;
};

// tile height and threads per CTA (a warp = TH / (NT / 32) tile rows)
template <int TH_, int NT_>
struct PairTGeom {
  static constexpr int TH = TH_, NT = NT_;
};

template <class MD, int STENCIL, int KA, int KB, class PG>
struct PairTShape {
  static constexpr int NV = MD::NV, ND = MD::ND, NG = NV - ND;
  static constexpr int R = stencil_radius(STENCIL);
  static constexpr int HX = 2;                         // x margin of the window: r rounded up to a pair
  static constexpr int TW = 64, TH = PG::TH, NT = PG::NT, NW = NT / 32;
  static constexpr int PW = TW / 2;                    // pairs per tile row = lanes
  static constexpr int WW = TW + 2 * HX, WPW = WW / 2, WH = TH + 2 * R, WSZ = WW * WH, TSZ = TW * TH;
  static constexpr int BW = TW + 4 * HX, BH = TH + 4 * R, BSZ = BW * BH;   // input box of a diffusing field
  static constexpr int NRING = 2 * R * WPW + 2 * TH;   // ring pairs: r rows above and below, one pair left and right
  // P1 slot
  static constexpr int OFF_INU = 0, SZ_INU = ND * BSZ * 8;
  static constexpr int OFF_ING = tma_align128(OFF_INU + SZ_INU), SZ_ING = NG * WSZ * 8;
  static constexpr int OFF_YU = tma_align128(OFF_ING + SZ_ING), SZ_YU = KA == K_BASE ? ND * WSZ * 8 : 0;
  static constexpr int OFF_YG = tma_align128(OFF_YU + SZ_YU), SZ_YG = KA == K_BASE ? NG * TSZ * 8 : 0;
  static constexpr int P1_BYTES = tma_align128(OFF_YG + SZ_YG);
  static constexpr unsigned TX1 = SZ_INU + SZ_ING + SZ_YU + SZ_YG;
  static constexpr bool HAS_P2 = KB == K_RK4F;
  static constexpr int P2_BYTES = HAS_P2 ? tma_align128(NV * TSZ * 8) : 0;
  static constexpr unsigned TX2 = HAS_P2 ? NV * TSZ * 8 : 0;
  static constexpr int NSLOT1 = KA == K_SELF ? 2 : 1;
  static constexpr int WIN_BYTES = tma_align128((ND * WSZ + (NG > 0 ? NG : 0) * TSZ) * 8);
  static constexpr int OFF_P2 = NSLOT1 * P1_BYTES, OFF_WIN = OFF_P2 + P2_BYTES, OFF_BAR = OFF_WIN + WIN_BYTES;
  static constexpr int SMEM_BYTES = OFF_BAR + 128;
  static_assert(TH % NW == 0 && NRING <= NT && R <= HX, "");
  static_assert(SMEM_BYTES <= 227 * 1024, "the slots of this instantiation do not fit one SM");
};

// Overwrite the ghost cells of a box — cells outside the grid, at most G beyond its edge — with the grid
// cell the index reflects / wraps to (rim tiles only).  box: [nf][bh][bw], its cell (0, 0) is grid cell
// (bx0, by0); src: field 0 of the same fields in global memory (batch member applied).  No-flux: the image
// of a ghost cell lies at most G inside the edge, i.e. inside the SAME box (every box reaches at least G
// inside the grid on the side it sticks out of), so the patch is shared memory -> shared memory; images
// are interior cells and ghost cells are never images, so no barrier is needed in between.  Periodic: the
// image is on the other side of the grid and is read from global memory.
template <int G>
CARDIAC_D void patch_box(double* __restrict__ box, int nf, int bw, int bh, int bx0, int by0,
                         const double* __restrict__ src, const Geom& g, int tid, int nt) {
  const int nx = g.nx, ny = g.ny, bc = g.boundary;
  auto image = [&](int q, int gx, int gy) -> double {   // (gx, gy) already reflected / wrapped into the grid
    if (bc == B_NOFLUX) return box[(q * bh + (gy - by0)) * bw + (gx - bx0)];
    return src[q * g.fstride + (long long)gy * g.pitch + gx];
  };
  if (bx0 < 0 || bx0 + bw > nx) {   // ghost columns -G..-1 and nx..nx+G-1, every box row whose image exists
    for (int e = tid; e < nf * bh * 2 * G; e += nt) {
      const int q = e / (bh * 2 * G), rr = (e / (2 * G)) % bh, k = e % (2 * G);
      const int gx = k < G ? -1 - k : nx + (k - G), gy = by0 + rr;
      const int cc = gx - bx0;
      if (cc >= 0 && cc < bw && gy >= -G && gy < ny + G)
        box[(q * bh + rr) * bw + cc] = image(q, bidx(gx, nx, bc), bidx(gy, ny, bc));
    }
  }
  if (by0 < 0 || by0 + bh > ny) {   // ghost rows -G..-1 and ny..ny+G-1 over the columns inside the grid
    for (int e = tid; e < nf * 2 * G * bw; e += nt) {
      const int q = e / (2 * G * bw), k = (e / bw) % (2 * G), cc = e % bw;
      const int gy = k < G ? -1 - k : ny + (k - G), gx = bx0 + cc;
      const int rr = gy - by0;
      if (rr >= 0 && rr < bh && gx >= 0 && gx < nx) box[(q * bh + rr) * bw + cc] = image(q, gx, bidx(gy, ny, bc));
    }
  }
}

// Substep KA of the pair at window position (wpx, wy), every operand from the P1 slot, no boundary logic.
// FULL: all fields (tile cells); otherwise the diffusing fields only (ring cells: the rest of the reaction
// is dead code).  Same instruction sequence per cell as pair_from_global (pair.cuh) / the stage kernels.
template <class MD, int STENCIL, int KA, int KB, class PG, bool FULL>
CARDIAC_D void pairt_substep_a(const PairTArgs<MD>& a, const unsigned char* __restrict__ slot, int wpx, int wy,
                               double2 (&res)[MD::NV]) {
  using S = PairTShape<MD, STENCIL, KA, KB, PG>;
  constexpr int NV = S::NV, ND = S::ND, NQ = FULL ? NV : ND, R = S::R, HX = S::HX;
  const double* inu = reinterpret_cast<const double*>(slot + S::OFF_INU);
  const double* ing = reinterpret_cast<const double*>(slot + S::OFF_ING);
  const double* yu = reinterpret_cast<const double*>(slot + S::OFF_YU);
  const double* yg = reinterpret_cast<const double*>(slot + S::OFF_YG);
  const int brow = (wy + R) * S::BW, bx = 2 * wpx + HX;   // the pair inside an input box
  const int wo = wy * S::WW + 2 * wpx;                     // ... inside a window box
  double2 zz[NV];
#pragma unroll
  for (int q = 0; q < ND; ++q) zz[q] = ld2(inu + q * S::BSZ + brow + bx);
#pragma unroll
  for (int q = ND; q < NV; ++q) zz[q] = ld2(ing + (q - ND) * S::WSZ + wo);
  double s0[ND], s1[ND];
#pragma unroll
  for (int q = 0; q < ND; ++q) stencil_pair<STENCIL>(inu + q * S::BSZ, brow, bx, S::BW, zz[q], s0[q], s1[q]);
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
#pragma unroll
  for (int q = 0; q < NQ; ++q) {
    double2 yy = make_double2(0.0, 0.0);
    if (KA != K_SELF)
      yy = q < ND ? ld2(yu + q * S::WSZ + wo) : ld2(yg + (q - ND) * S::TSZ + (wy - R) * S::TW + 2 * wpx - HX);
    res[q].x = combine<KA>(a.a_wy, a.a_win, 0.0, 0.0, a.a_wf, yy.x, z0[q], 0.0, 0.0, f0[q]);
    res[q].y = combine<KA>(a.a_wy, a.a_win, 0.0, 0.0, a.a_wf, yy.y, z1[q], 0.0, 0.0, f1[q]);
  }
}

template <class MD, int STENCIL, int KA, int KB, bool WRITE_P, class PG>
__global__ void __launch_bounds__(PG::NT, 1)
    pair_tma_kernel(const __grid_constant__ PairTArgs<MD> a, const __grid_constant__ CUtensorMap tm_inu,
                    const __grid_constant__ CUtensorMap tm_ing, const __grid_constant__ CUtensorMap tm_yu,
                    const __grid_constant__ CUtensorMap tm_yg, const __grid_constant__ CUtensorMap tm_p) {
  using S = PairTShape<MD, STENCIL, KA, KB, PG>;
  constexpr int NV = S::NV, ND = S::ND, NG = S::NG, R = S::R, HX = S::HX, TW = S::TW, TH = S::TH;
  constexpr int WW = S::WW, WPW = S::WPW, WH = S::WH, WSZ = S::WSZ, TSZ = S::TSZ, NT = S::NT, NW = S::NW;
  constexpr int NSLOT1 = S::NSLOT1;
  static_assert(!(WRITE_P && !(KA == K_SELF && KB == K_BASE)), "P is formed by RK4 launch 1");
  extern __shared__ __align__(1024) unsigned char pt_smem[];
  unsigned char* const p2 = pt_smem + S::OFF_P2;
  double* const sw = reinterpret_cast<double*>(pt_smem + S::OFF_WIN);   // [ND][WH][WW]
  double* const sg = sw + ND * WSZ;                                      // [NG][TH][TW]
  uint64_t* const full1 = reinterpret_cast<uint64_t*>(pt_smem + S::OFF_BAR);
  uint64_t* const full2 = full1 + NSLOT1;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int nx = a.g.nx, ny = a.g.ny, pitch = a.g.pitch;

  // the box copies of tile t (one elected thread)
  auto issue1 = [&](unsigned t, int s) {
    const TilePos tp = tile_pos_of(t, a.per_member, a.per_row, a.tiles_x, TW, TH);
    unsigned char* slot = pt_smem + s * S::P1_BYTES;
    mbar_arrive_expect_tx(full1 + s, S::TX1);
    tma_load_4d(slot + S::OFF_INU, &tm_inu, tp.x0 - 2 * HX, tp.y0 - 2 * R, 0, tp.bz, full1 + s);
    if (NG > 0) tma_load_4d(slot + S::OFF_ING, &tm_ing, tp.x0 - HX, tp.y0 - R, 0, tp.bz, full1 + s);
    if (KA == K_BASE) {
      tma_load_4d(slot + S::OFF_YU, &tm_yu, tp.x0 - HX, tp.y0 - R, 0, tp.bz, full1 + s);
      if (NG > 0) tma_load_4d(slot + S::OFF_YG, &tm_yg, tp.x0, tp.y0, 0, tp.bz, full1 + s);
    }
  };
  auto issue2 = [&](unsigned t) {
    const TilePos tp = tile_pos_of(t, a.per_member, a.per_row, a.tiles_x, TW, TH);
    mbar_arrive_expect_tx(full2, S::TX2);
    tma_load_4d(p2, &tm_p, tp.x0, tp.y0, 0, tp.bz, full2);
  };

  if (tid == 0) {
#pragma unroll
    for (int s = 0; s < NSLOT1 + 1; ++s) mbar_init(full1 + s, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  }
  __syncthreads();
  // programmatic dependent launch: everything above overlaps the tail of the previous launch; every
  // global access below (TMA included) waits for that grid to complete and flush
  asm volatile("griddepcontrol.wait;" ::: "memory");
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  if (tid == 0) {
    unsigned t = blockIdx.x;
#pragma unroll
    for (int s = 0; s < NSLOT1; ++s, t += gridDim.x)
      if (t < a.ntiles) issue1(t, s);
    if (S::HAS_P2 && blockIdx.x < a.ntiles) issue2(blockIdx.x);
  }

  int s1 = 0;
  unsigned ph1 = 0, ph2 = 0;
  for (unsigned t = blockIdx.x; t < a.ntiles; t += gridDim.x) {
    const TilePos tp = tile_pos_of(t, a.per_member, a.per_row, a.tiles_x, TW, TH);
    const int x0 = tp.x0, y0 = tp.y0;
    const long long base = (long long)tp.bz * a.g.bstride;
    unsigned char* const slot = pt_smem + s1 * S::P1_BYTES;
    mbar_wait(full1 + s1, ph1);

    // ------------------------------------------------------------ rim tiles: even / periodic extension
    if (x0 < 2 * HX || x0 + TW + 2 * HX > nx || y0 < 2 * R || y0 + TH + 2 * R > ny) {
      patch_box<2 * R>(reinterpret_cast<double*>(slot + S::OFF_INU), ND, S::BW, S::BH, x0 - 2 * HX, y0 - 2 * R,
                       a.in + base, a.g, tid, NT);
      if (NG > 0)
        patch_box<R>(reinterpret_cast<double*>(slot + S::OFF_ING), NG, WW, WH, x0 - HX, y0 - R,
                     a.in + base + ND * a.g.fstride, a.g, tid, NT);
      if (KA == K_BASE)
        patch_box<R>(reinterpret_cast<double*>(slot + S::OFF_YU), ND, WW, WH, x0 - HX, y0 - R, a.y + base, a.g, tid, NT);
      asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // generic writes before the next TMA write
      __syncthreads();
    }

    // ------------------------------------------------------------ phase 1: substep A -> shared window
#pragma unroll 1
    for (int py = warp; py < TH; py += NW) {   // tile cells: every field
      if (y0 + py > ny - 1 + R) break;          // beyond the ghost rows of a ragged tile
      double2 res[NV];
      pairt_substep_a<MD, STENCIL, KA, KB, PG, true>(a, slot, lane + HX / 2, py + R, res);
#pragma unroll
      for (int q = 0; q < NV; ++q) {
        if (q < ND) *reinterpret_cast<double2*>(sw + q * WSZ + (py + R) * WW + HX + 2 * lane) = res[q];
        else *reinterpret_cast<double2*>(sg + (q - ND) * TSZ + py * TW + 2 * lane) = res[q];
      }
    }
    if (tid < S::NRING) {   // ring cells: the diffusing fields only
      int wy, wpx;
      if (tid < 2 * R * WPW) {
        const int rr = tid / WPW;
        wpx = tid - rr * WPW;
        wy = rr < R ? rr : TH + rr;
      } else {
        const int r2 = tid - 2 * R * WPW;
        wy = R + (r2 >> 1);
        wpx = (r2 & 1) ? WPW - 1 : 0;
      }
      if (y0 - R + wy <= ny - 1 + R) {
        double2 res[NV];
        pairt_substep_a<MD, STENCIL, KA, KB, PG, false>(a, slot, wpx, wy, res);
#pragma unroll
        for (int q = 0; q < ND; ++q) *reinterpret_cast<double2*>(sw + q * WSZ + wy * WW + 2 * wpx) = res[q];
      }
    }
    __syncthreads();   // the window is complete; nobody reads the phase-1 operands any more (KA = K_BASE)
    if (KA == K_BASE && tid == 0) {
      const unsigned long long tn = (unsigned long long)t + gridDim.x;
      if (tn < a.ntiles) issue1((unsigned)tn, 0);   // in flight during phase 2
    }

    // ------------------------------------------------------------ phase 2: substep B, tile cells
    if (S::HAS_P2) mbar_wait(full2, ph2);
    {
      const int x = x0 + 2 * lane;
      const bool both = x + 1 < nx;
      const int rows = min(TH, ny - y0);
      double* const ob = a.out + base + x;
      double* const ob2 = a.out2 + base + x;
      const double* inu = reinterpret_cast<const double*>(slot + S::OFF_INU);
      const double* ing = reinterpret_cast<const double*>(slot + S::OFF_ING);
      const double* ps = reinterpret_cast<const double*>(p2);
#pragma unroll 1
      for (int py = warp; py < rows; py += NW) {
        if (x >= nx) break;
        const int srow = (py + R) * WW, sx = HX + 2 * lane;
        double2 zz[NV];
#pragma unroll
        for (int q = 0; q < NV; ++q)
          zz[q] = q < ND ? ld2(sw + q * WSZ + srow + sx) : ld2(sg + (q - ND) * TSZ + py * TW + 2 * lane);
        double s0[ND], s1v[ND];
#pragma unroll
        for (int q = 0; q < ND; ++q) stencil_pair<STENCIL>(sw + q * WSZ, srow, sx, WW, zz[q], s0[q], s1v[q]);
        double z0[NV], z1[NV], f0[NV], f1[NV];
#pragma unroll
        for (int q = 0; q < NV; ++q) { z0[q] = zz[q].x; z1[q] = zz[q].y; }
        MD::reaction(a.p, z0, f0);
        MD::reaction(a.p, z1, f1);
#pragma unroll
        for (int q = 0; q < ND; ++q) {
          f0[q] = fma(a.lapw[q], s0[q], f0[q]);
          f1[q] = fma(a.lapw[q], s1v[q], f1[q]);
        }
        const int o = (y0 + py) * pitch;
#pragma unroll
        for (int q = 0; q < NV; ++q) {
          double2 yy = make_double2(0.0, 0.0);
          if (S::HAS_P2) {
            yy = ld2(ps + q * TSZ + py * TW + 2 * lane);
          } else if (KB != K_SELF) {   // y = the input of substep A, still in the P1 slot
            yy = q < ND ? ld2(inu + q * S::BSZ + (py + 2 * R) * S::BW + 2 * HX + 2 * lane)
                        : ld2(ing + (q - ND) * WSZ + (py + R) * WW + HX + 2 * lane);
          }
          double r0, r1;
          if (S::HAS_P2) {   // = combine<K_RK4F> with its inner part P formed by launch 1
            r0 = fma(a.w_f, f0[q], fma(a.w_in, z0[q], yy.x));
            r1 = fma(a.w_f, f1[q], fma(a.w_in, z1[q], yy.y));
          } else {
            r0 = combine<KB>(a.w_y, a.w_in, 0.0, 0.0, a.w_f, yy.x, z0[q], 0.0, 0.0, f0[q]);
            r1 = combine<KB>(a.w_y, a.w_in, 0.0, 0.0, a.w_f, yy.y, z1[q], 0.0, 0.0, f1[q]);
          }
          if (both) st2(ob + o + q * a.g.fstride, r0, r1);
          else ob[o + q * a.g.fstride] = r0;
          if (WRITE_P) {   // the inner part of combine<K_RK4F>: w_B B + (w_A A + w_y y), A = Y2, B = Y3
            const double p0 = fma(a.p_wB, r0, fma(a.p_wA, z0[q], a.p_wy * yy.x));
            const double p1 = fma(a.p_wB, r1, fma(a.p_wA, z1[q], a.p_wy * yy.y));
            if (both) st2(ob2 + o + q * a.g.fstride, p0, p1);
            else ob2[o + q * a.g.fstride] = p0;
          }
        }
      }
    }
    __syncthreads();   // the window and this tile's slots are free
    if (tid == 0) {
      if (S::HAS_P2) {
        const unsigned long long tn = (unsigned long long)t + gridDim.x;
        if (tn < a.ntiles) issue2((unsigned)tn);      // in flight during the next phase 1
      }
      if (KA == K_SELF) {
        const unsigned long long tn = (unsigned long long)t + (unsigned long long)NSLOT1 * gridDim.x;
        if (tn < a.ntiles) issue1((unsigned)tn, s1);
      }
    }
    ph2 ^= 1;
    if (++s1 == NSLOT1) { s1 = 0; ph1 ^= 1; }
  }
}

}  // namespace cardiac
