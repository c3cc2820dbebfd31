// pair.cuh — plan PAIR: TWO consecutive RK substeps per launch.
//
// The stage-synchronous plan pays one global round trip per substep (the paper's lock-step,
// PAPER.md:130-134); the on-chip tile engine (tile.cuh) pays one per time step but keeps every field of
// its window in registers, which the 4-field ionic model cannot afford.  This plan
// sits between the two.  A CTA owns a tile of TW x TH cells:
//
//   phase 1  substep A on the tile PLUS a ring of r cells, operands from global memory (stencil
//            neighbours through L1, exactly as the DIRECT stage kernel).  The result stays in shared
//            memory: a window (TW+4) x (TH+2r) of every DIFFUSING field, and the gating fields on the
//            tile only — the ring exists to feed the stencil of substep B, so ring cells evaluate
//            the right-hand side of the diffusing fields alone (for BOCF: the currents, 1 of the 3
//            exponentials and 2 of the 5 reciprocals of a full cell).
//   phase 2  substep B on the tile, stencil and reaction input from shared memory, ONE pointwise RK
//            operand per field from global memory, result to global memory.
//
// RK4, accumulator-free (same combinations, same weights and hence the same bits as plan STAGE):
//   launch 1:  Y2 = y + dt/2 f(y)  [shared + global],   Y3 = y + dt/2 f(Y2)                 [global]
//   launch 2:  Y4 = y + dt f(Y3)   [shared only],       y+ = (Y2 + 2 Y3 + Y4 - y)/3 + dt/6 f(Y4)
// (phase 1 of launch 2 also forms P = (2 Y3 + Y2 - y)/3, the part of y+ that does not depend on Y4,
// and leaves it where y+ will be written), i.e. 4 + 8 and 12 + 4 doubles per cell and field instead of
// 52: 224 B instead of 416 B per cell-step for the 4-field model.  Heun is ONE launch (Y2 never leaves
// the SM), forward Euler two time steps per launch (temporal blocking, north_star).
//
// Boundary (PAPER.md:104 Fig. 1, :114): a ring cell outside the grid is the image of the grid cell the
// index reflects (or wraps) to; rim tiles evaluate substep A AT that image with the boundary rule
// applied per neighbour and store the value at the ghost position, so that phase 2 has no boundary
// logic.  Every value is produced by the same instruction sequence wherever it is evaluated, so the
// result does not depend on the tiling.
#pragma once
#include "plans.h"
#include "stage.cuh"

namespace cardiac {

template <class MD>
struct PairArgs {
  const double* in;   // input of substep A (global; diffusing fields read with halo 2r)
  const double* y;    // state at the start of the time step (pointwise, both substeps)
  const double* A;    // Y2 (pointwise, substep B = K_RK4F)
  const double* B;    // Y3 (substep B = K_RK4F): must be `in`, the input of substep A
  double* mid;        // where the tile cells of substep A's result are also stored, if they are
  double* out;        // result of substep B; never `in` or `y` (other CTAs read their halos), may be `A`
  Geom g;
  double a_wy, a_win, a_wf;            // substep A: K_SELF in + a_wf f(in), K_BASE a_wy y + a_win in + a_wf f(in)
  double w_y, w_in, w_A, w_B, w_f;     // substep B, as StageArgs
  double lapw[MD::ND];
  typename MD::Params p;
};

template <int TW_, int TH_, int NT_, int MINB_>
struct PairGeom {
  static constexpr int TW = TW_, TH = TH_, NT = NT_, MINB = MINB_;
};

template <class MD, int STENCIL, class PG>
struct PairShape {
  static constexpr int NV = MD::NV, ND = MD::ND, NG = NV - ND;
  static constexpr int R = stencil_radius(STENCIL);
  static constexpr int HX = 2;                        // x halo of the window: r rounded up to a pair
  static constexpr int TW = PG::TW, TH = PG::TH;
  static constexpr int PW = TW / 2;                   // pairs per tile row
  static constexpr int WW = TW + 2 * HX, WPW = WW / 2, WH = TH + 2 * R;
  static constexpr int WSZ = WW * WH, TSZ = TW * TH;  // doubles per windowed / per tile-only field
  static constexpr int NBODY = PW * TH;               // pairs of the tile
  static constexpr int NRING = 2 * R * WPW + 2 * TH;  // pairs of the ring: r rows above and below, one pair left and right
  static constexpr int NWIN = WPW * WH;
  static constexpr int SMEM_BYTES = (ND * WSZ + (NG > 0 ? NG : 0) * TSZ) * (int)sizeof(double);
  static_assert(TW % 2 == 0 && R <= HX, "");
};

// a 128-bit global load the compiler may not sink towards its use
CARDIAC_D double2 ld2v(const double* p) {
  double2 v;
  asm volatile("ld.global.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "l"(p));
  return v;
}

// Substep KIND of the x-adjacent pair at (x, row/pitch), every operand from global memory, no boundary
// logic.  FULL: all fields; otherwise the diffusing fields only (the rest of the reaction is dead code).
// PRE (substep B = K_RK4F, tile cells): also forms the part of the final combination that does not
// depend on substep B's result, P = w_B Y3 + (w_A Y2 + w_y y) — Y3 is this substep's input — and
// stores it where substep B will write (which may be where Y2 was read: same thread, same cell).
// BC: the pair lies inside the grid but its stencil may reach across the boundary (stencil_pair_bc).
template <class MD, int STENCIL, int KIND, bool FULL, bool PRE, bool EARLY = false, bool BC = false>
CARDIAC_D void pair_from_global(const PairArgs<MD>& a, const double* __restrict__ in,
                                const double* __restrict__ yb, const double* Ab, double* ob, int row, int x,
                                double2 (&res)[MD::NV]) {
  constexpr int NV = MD::NV, ND = MD::ND, NQ = FULL ? NV : ND;
  const int o = row + x;
  if (NV > 2) {   // see stage_kernels.cu: the late operands are asked for now, at no register cost
#pragma unroll
    for (int q = ND; q < NV; ++q) prefetch_l1(in + o + q * a.g.fstride);
  }
  if (KIND == K_BASE) {
#pragma unroll
    for (int q = 0; q < NQ; ++q) prefetch_l1(yb + o + q * a.g.fstride);
  }
  double2 zz[NV];
#pragma unroll
  for (int q = 0; q < NV; ++q) zz[q] = ld2(in + o + q * a.g.fstride);
  double s0[ND], s1[ND];
#pragma unroll
  for (int q = 0; q < ND; ++q) {
    if (BC) stencil_pair_bc<STENCIL>(in + q * a.g.fstride, x, row / a.g.pitch, a.g.nx, a.g.ny, a.g.pitch, a.g.boundary, zz[q], s0[q], s1[q]);
    else stencil_pair<STENCIL>(in + q * a.g.fstride, row, x, a.g.pitch, zz[q], s0[q], s1[q]);
  }
  // EARLY (tile cells of interior tiles): every global operand of the row is requested before the
  // reaction starts, so that a warp waits for memory once per row; costs 8 registers per operand
  double2 yy[NV], AA[NV];
  if (EARLY) {
#pragma unroll
    for (int q = 0; q < NQ; ++q) {
      if (KIND != K_SELF) yy[q] = ld2v(yb + o + q * a.g.fstride);
      if (PRE) AA[q] = ld2v(Ab + o + q * a.g.fstride);
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
#pragma unroll
  for (int q = 0; q < NQ; ++q) {
    if (!EARLY) {
      yy[q] = make_double2(0.0, 0.0);
      if (KIND != K_SELF) yy[q] = ld2(yb + o + q * a.g.fstride);
      if (PRE) AA[q] = ld2(Ab + o + q * a.g.fstride);
    }
    res[q].x = combine<KIND>(a.a_wy, a.a_win, 0.0, 0.0, a.a_wf, yy[q].x, z0[q], 0.0, 0.0, f0[q]);
    res[q].y = combine<KIND>(a.a_wy, a.a_win, 0.0, 0.0, a.a_wf, yy[q].y, z1[q], 0.0, 0.0, f1[q]);
    if (PRE) {
      st2(ob + o + q * a.g.fstride, fma(a.w_B, z0[q], fma(a.w_A, AA[q].x, a.w_y * yy[q].x)),
          fma(a.w_B, z1[q], fma(a.w_A, AA[q].y, a.w_y * yy[q].y)));
    }
  }
}

// ... of ONE window cell: evaluated at grid cell (i, j) — the cell itself or the one it is the image
// of — with the boundary rule applied per neighbour
template <class MD, int STENCIL, int KIND, bool FULL, bool PRE>
CARDIAC_D void cell_from_global(const PairArgs<MD>& a, const double* __restrict__ in,
                                const double* __restrict__ yb, const double* Ab, double* ob, int i, int j,
                                double (&res)[MD::NV]) {
  constexpr int NV = MD::NV, ND = MD::ND, NQ = FULL ? NV : ND;
  const int o = j * a.g.pitch + i;
  double z[NV], f[NV];
#pragma unroll
  for (int q = 0; q < NV; ++q) z[q] = in[o + q * a.g.fstride];
  MD::reaction(a.p, z, f);
#pragma unroll
  for (int q = 0; q < ND; ++q) {
    const double s = stencil_edge<STENCIL>(in + q * a.g.fstride, i, j, a.g.nx, a.g.ny, a.g.pitch, a.g.boundary, z[q]);
    f[q] = fma(a.lapw[q], s, f[q]);
  }
#pragma unroll
  for (int q = 0; q < NQ; ++q) {
    const double yv = KIND != K_SELF ? yb[o + q * a.g.fstride] : 0.0;
    res[q] = combine<KIND>(a.a_wy, a.a_win, 0.0, 0.0, a.a_wf, yv, z[q], 0.0, 0.0, f[q]);
    if (PRE) ob[o + q * a.g.fstride] = fma(a.w_B, z[q], fma(a.w_A, Ab[o + q * a.g.fstride], a.w_y * yv));
  }
}

// Phase 1 of a tile that touches the rim of the grid (or is ragged): the same two passes, but every
// pair decides for itself whether it and its stencil arms lie inside the grid (128-bit path) or its
// cells are evaluated one by one with the boundary rule, ghost cells at their images.  Kept out of line
// so that its registers do not weigh on the interior path.
template <class MD, int STENCIL, int KA, bool PRE, bool STORE_MID, class PG>
__device__ __noinline__ void pair_phase1_rim(const PairArgs<MD>& a, double* __restrict__ sw,
                                             double* __restrict__ sg, int x0, int y0, long long base) {
  using S = PairShape<MD, STENCIL, PG>;
  constexpr int NV = S::NV, ND = S::ND, R = S::R, HX = S::HX, TW = S::TW, TH = S::TH, PW = S::PW;
  constexpr int WW = S::WW, WPW = S::WPW, WSZ = S::WSZ, TSZ = S::TSZ, NT = PG::NT;
  const int nx = a.g.nx, ny = a.g.ny, pitch = a.g.pitch, bc = a.g.boundary;
  const double* __restrict__ in = a.in + base;
  const double* __restrict__ yb = a.y + base;
  const double* Ab = a.A + base;
  double* mid = a.mid + base;
  double* ob = a.out + base;
#pragma unroll 1
  for (int it = threadIdx.x; it < S::NBODY + S::NRING; it += NT) {
    const bool body = it < S::NBODY;
    int wy, wpx;
    if (body) {
      wy = it / PW;
      wpx = it - wy * PW + HX / 2;
      wy += R;
    } else {
      const int r = it - S::NBODY;
      if (r < 2 * R * WPW) {
        const int rr = r / WPW;
        wpx = r - rr * WPW;
        wy = rr < R ? rr : TH + rr;
      } else {
        const int r2 = r - 2 * R * WPW;
        wy = R + (r2 >> 1);
        wpx = (r2 & 1) ? WPW - 1 : 0;
      }
    }
    const int x = x0 - HX + 2 * wpx, j = y0 - R + wy;
    if (x > nx - 1 + R || j > ny - 1 + R) continue;   // beyond the ghost cells of a ragged tile
    double* const swp = sw + wy * WW + 2 * wpx;
    double* const sgp = sg + (wy - R) * TW + 2 * wpx - HX;   // body only
    if (x >= 2 && x + 4 <= nx && j >= R && j + R < ny) {
      double2 res[NV];
      if (body) {
        pair_from_global<MD, STENCIL, KA, true, PRE>(a, in, yb, Ab, ob, j * pitch, x, res);
#pragma unroll
        for (int q = ND; q < NV; ++q) *reinterpret_cast<double2*>(sgp + (q - ND) * TSZ) = res[q];
        if (STORE_MID) {
#pragma unroll
          for (int q = 0; q < NV; ++q) st2(mid + j * pitch + x + q * a.g.fstride, res[q].x, res[q].y);
        }
      } else {
        pair_from_global<MD, STENCIL, KA, false, false>(a, in, yb, Ab, ob, j * pitch, x, res);
      }
#pragma unroll
      for (int q = 0; q < ND; ++q) *reinterpret_cast<double2*>(swp + q * WSZ) = res[q];
    } else if (x >= 0 && x + 1 < nx && j >= 0 && j < ny) {
      // inside the grid, its stencil across the boundary: still 128-bit loads
      double2 res[NV];
      if (body) {
        pair_from_global<MD, STENCIL, KA, true, PRE, false, true>(a, in, yb, Ab, ob, j * pitch, x, res);
#pragma unroll
        for (int q = ND; q < NV; ++q) *reinterpret_cast<double2*>(sgp + (q - ND) * TSZ) = res[q];
        if (STORE_MID) {
#pragma unroll
          for (int q = 0; q < NV; ++q) st2(mid + j * pitch + x + q * a.g.fstride, res[q].x, res[q].y);
        }
      } else {
        pair_from_global<MD, STENCIL, KA, false, false, false, true>(a, in, yb, Ab, ob, j * pitch, x, res);
      }
#pragma unroll
      for (int q = 0; q < ND; ++q) *reinterpret_cast<double2*>(swp + q * WSZ) = res[q];
    } else {
#pragma unroll 1
      for (int h = 0; h < 2; ++h) {
        const int cx = x + h;
        if (cx < -R || cx > nx - 1 + R || j < -R) continue;
        double res[NV];
        if (body && cx < nx && j < ny) {
          cell_from_global<MD, STENCIL, KA, true, PRE>(a, in, yb, Ab, ob, cx, j, res);
#pragma unroll
          for (int q = ND; q < NV; ++q) sgp[(q - ND) * TSZ + h] = res[q];
          if (STORE_MID) {
#pragma unroll
            for (int q = 0; q < NV; ++q) mid[j * pitch + cx + q * a.g.fstride] = res[q];
          }
        } else {   // a ring cell, or a ghost cell inside a ragged tile: the diffusing fields, at the image
          cell_from_global<MD, STENCIL, KA, false, false>(a, in, yb, Ab, ob, bidx(cx, nx, bc), bidx(j, ny, bc), res);
        }
#pragma unroll
        for (int q = 0; q < ND; ++q) swp[q * WSZ + h] = res[q];
      }
    }
  }
}

template <class MD, int STENCIL, int KA, int KB, bool STORE_MID, class PG>
__global__ void __launch_bounds__(PG::NT, PG::MINB)
    pair_kernel(const __grid_constant__ PairArgs<MD> a) {
  using S = PairShape<MD, STENCIL, PG>;
  constexpr int NV = S::NV, ND = S::ND, R = S::R, HX = S::HX, TW = S::TW, TH = S::TH, PW = S::PW;
  constexpr int WW = S::WW, WPW = S::WPW, WSZ = S::WSZ, TSZ = S::TSZ, NT = PG::NT;
  constexpr int RSTEP = NT / PW;            // tile rows one pass of the CTA covers
  constexpr bool PRE = KB == K_RK4F;
  static_assert(NT % PW == 0 && S::NRING <= NT, "");
  extern __shared__ double2 smem_pair[];
  double* const sw = reinterpret_cast<double*>(smem_pair);   // [ND][WH][WW]
  double* const sg = sw + ND * WSZ;                          // [NG][TH][TW]

  const int nx = a.g.nx, ny = a.g.ny, pitch = a.g.pitch;
  const int x0 = blockIdx.x * TW, y0 = blockIdx.y * TH;
  const long long base = (long long)blockIdx.z * a.g.bstride;
  const int tid = threadIdx.x;
  const int py0 = tid / PW, px = tid - py0 * PW;   // a thread keeps its column pair; rows py0, py0 + RSTEP, ...
  // programmatic dependent launch: this grid may be scheduled while the previous launch drains; every
  // global access below waits for that grid to complete and flush
  asm volatile("griddepcontrol.wait;" ::: "memory");
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");

  // ---------------------------------------------------------------- phase 1: substep A -> shared memory
  // block-uniform: the window and the stencil arms of its outermost cells lie inside the grid
  const bool interior = x0 >= 4 && x0 + TW + 4 <= nx && y0 >= 2 * R && y0 + TH + 2 * R <= ny;
  if (interior) {
    {
      const double* __restrict__ in = a.in + base;
      const double* __restrict__ yb = a.y + base;
      const double* Ab = a.A + base;   // may alias out
      double* ob = a.out + base;
      const int x = x0 + 2 * px;
#pragma unroll 1
      for (int py = py0; py < TH; py += RSTEP) {   // tile cells: every field
        const int row = (y0 + py) * pitch;
        if (py + RSTEP < TH) {   // the operands of this thread's next row: towards L1 while this row computes
          const int on = row + RSTEP * pitch + x;
#pragma unroll
          for (int q = 0; q < NV; ++q) {
            prefetch_l1(in + on + q * a.g.fstride);
            if (KA == K_BASE) prefetch_l1(yb + on + q * a.g.fstride);
            if (PRE) prefetch_l1(Ab + on + q * a.g.fstride);
          }
        }
        double2 res[NV];
        pair_from_global<MD, STENCIL, KA, true, PRE, true>(a, in, yb, Ab, ob, row, x, res);
#pragma unroll
        for (int q = 0; q < NV; ++q) {
          if (q < ND) *reinterpret_cast<double2*>(sw + q * WSZ + (py + R) * WW + HX + 2 * px) = res[q];
          else *reinterpret_cast<double2*>(sg + (q - ND) * TSZ + py * TW + 2 * px) = res[q];
          if (STORE_MID) st2(a.mid + base + row + x + q * a.g.fstride, res[q].x, res[q].y);
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
        double2 res[NV];
        pair_from_global<MD, STENCIL, KA, false, false>(a, in, yb, Ab, ob, (y0 - R + wy) * pitch, x0 - HX + 2 * wpx, res);
#pragma unroll
        for (int q = 0; q < ND; ++q) *reinterpret_cast<double2*>(sw + q * WSZ + wy * WW + 2 * wpx) = res[q];
      }
    }
  } else {
    pair_phase1_rim<MD, STENCIL, KA, PRE, STORE_MID, PG>(a, sw, sg, x0, y0, base);
  }
  __syncthreads();

  // ---------------------------------------------------------------- phase 2: substep B, tile cells
  const int x = x0 + 2 * px;
  if (x >= nx) return;
  const bool both = x + 1 < nx;
  const int rows = min(TH, ny - y0);
  // the pointwise operand of the combination: y, or (K_RK4F) the P that phase 1 left in `out`
  double* const ob = a.out + base + x;
  const double* const pb = PRE ? ob : a.y + base + x;
#pragma unroll 1
  for (int py = py0; py < rows; py += RSTEP) {
    const int o = (y0 + py) * pitch;
    double2 yq[NV];
    if (KB != K_SELF) {   // this row's operand now (used after the reaction), the next row's towards L1
#pragma unroll
      for (int q = 0; q < NV; ++q) {
        if (py + RSTEP < rows) prefetch_l1(pb + o + RSTEP * pitch + q * a.g.fstride);
        yq[q] = ld2v(pb + o + q * a.g.fstride);
      }
    }
    const int srow = (py + R) * WW, sx = HX + 2 * px;
    double2 zz[NV];
#pragma unroll
    for (int q = 0; q < NV; ++q)
      zz[q] = q < ND ? ld2(sw + q * WSZ + srow + sx) : ld2(sg + (q - ND) * TSZ + py * TW + 2 * px);
    double s0[ND], s1[ND];
#pragma unroll
    for (int q = 0; q < ND; ++q) stencil_pair<STENCIL>(sw + q * WSZ, srow, sx, WW, zz[q], s0[q], s1[q]);
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
    for (int q = 0; q < NV; ++q) {
      const double2 yy = KB != K_SELF ? yq[q] : make_double2(0.0, 0.0);
      double r0, r1;
      if (PRE) {   // = combine<K_RK4F> with its inner part already formed
        r0 = fma(a.w_f, f0[q], fma(a.w_in, z0[q], yy.x));
        r1 = fma(a.w_f, f1[q], fma(a.w_in, z1[q], yy.y));
      } else {
        r0 = combine<KB>(a.w_y, a.w_in, 0.0, 0.0, a.w_f, yy.x, z0[q], 0.0, 0.0, f0[q]);
        r1 = combine<KB>(a.w_y, a.w_in, 0.0, 0.0, a.w_f, yy.y, z1[q], 0.0, 0.0, f1[q]);
      }
      if (both) st2(ob + o + q * a.g.fstride, r0, r1);
      else ob[o + q * a.g.fstride] = r0;
    }
  }
}

}  // namespace cardiac
