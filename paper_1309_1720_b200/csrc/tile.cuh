// tile.cuh — the on-chip tile engine behind plan FUSED.
//
// One CTA advances one tile of the grid through ALL substeps of a time step (or through several
// Euler steps) without leaving the SM: the paper's lock-step, one global round trip per substep
// (PAPER.md:130-134), becomes one round trip per time step.  The price is the classic overlapped
// ("trapezoid") tiling: a tile of TW x TH output cells is loaded with a halo of H = r * n_stages
// cells, and substep s is evaluated on the region that is still r*(s+1) cells inside the loaded
// window.  Halo cells are recomputed by the neighbouring tiles; they go through exactly the same
// instruction sequence on the same inputs, so the result does not depend on the tiling.
//
// Boundary (PAPER.md:104 Fig. 1, :114): the window of a rim tile reaches outside the grid.  It is
// filled, at load time, from the mirrored (or wrapped) cell — the even extension of the grid about
// its boundary nodes — and the ghost cells are then advanced like any other cell.  The stencils are
// reflection symmetric and written as sums of (west+east), (south+north) pairs, so a ghost cell
// reproduces its mirror image bitwise and no boundary logic is left inside the stage loop: this is
// the paper's "pre-populated ghost ring" alternative generalised to H rings.
//
// Data placement (north_star: "shared-memory tile staging of the u halo, register-resident gating
// variables"): only the stage value of the DIFFUSING fields lives in shared memory (two buffers,
// read with 128-bit LDS); each thread owns a fixed 2 x PR patch of cells and keeps their step-start
// value y, the running RK sum and the non-diffusing (gating) variables in registers for the whole
// step.  y-neighbours are reused through a rolling register window of 2r+1 rows.
#pragma once
#include "stage.cuh"

namespace cardiac {

// substeps per launch and whether the RK bookkeeping (y, acc) is needed
template <int INTEG, int KSTEPS>
struct StepScheme {
  static constexpr int NS = INTEG == I_RK4 ? 4 : (INTEG == I_HEUN ? 2 : KSTEPS);
  static constexpr bool RK = INTEG != I_EULER;
};

template <int NTX_, int NTY_, int PR_, int MINB_ = 1>
struct TileGeom {
  static constexpr int NTX = NTX_, NTY = NTY_, PR = PR_;
  static constexpr int MINB = MINB_;  // CTAs per SM the register budget is held to
  static constexpr int NT = NTX * NTY;
  static constexpr int EW = 2 * NTX, EH = PR * NTY;  // loaded window
};

template <class MD>
struct TileArgs {
  const double* in;
  double* out;
  Geom g;
  double a_dt[4];  // next stage value  = y   + a_dt[s] f   (Euler: cur + a_dt[0] f)
  double b_dt[4];  // running sum       = acc + b_dt[s] f   (acc starts at y)
  double lapw[MD::ND];
  typename MD::Params p;
};

// index of the grid cell that the even (no-flux) or periodic extension maps `i` to; any i
CARDIAC_D int fold(int i, int n, int boundary) {
  if (boundary == B_PERIODIC) {
    i %= n;
    return i < 0 ? i + n : i;
  }
  const int period = 2 * (n - 1);
  i %= period;
  if (i < 0) i += period;
  return i < n ? i : period - i;
}

template <class MD, int STENCIL, int INTEG, int KSTEPS, class TG>
struct TileEngine {
  static constexpr int NV = MD::NV, ND = MD::ND, NG = NV - ND;
  static constexpr int R = stencil_radius(STENCIL);
  static constexpr int NS = StepScheme<INTEG, KSTEPS>::NS;
  static constexpr bool RK = StepScheme<INTEG, KSTEPS>::RK;
  static constexpr int H = R * NS;
  static constexpr int PR = TG::PR, NTX = TG::NTX, EW = TG::EW, EH = TG::EH;
  static constexpr int TW = EW - 2 * H, TH = EH - 2 * H;  // output tile
  static constexpr int PADX = 2;                          // keeps every pair 16-byte aligned
  static constexpr int SP = EW + 2 * PADX;                // shared row pitch, doubles
  static constexpr int SR = EH + 2 * R;                   // shared rows
  static constexpr int FSZ = SP * SR;                     // one field, one buffer
  static constexpr int SMEM_BYTES = 2 * ND * FSZ * (int)sizeof(double);
  static constexpr bool VEC = (H % 2 == 0);               // window pairs are 16-byte aligned in global memory
  static_assert(TW > 0 && TH > 0 && TW % 2 == 0, "tile too small for its halo");
  static_assert(NG >= 0 && PR >= 1, "");

  // per-thread state of the 2 x PR patch
  struct Patch {
    double y[RK ? PR : 1][2][NV];
    double acc[RK ? PR : 1][2][NV];
    double g[PR][2][NG > 0 ? NG : 1];
  };

  CARDIAC_D static double2 lds2(const double* p) { return *reinterpret_cast<const double2*>(p); }

  // Load the window of tile (bx, by) of batch member `in` (already offset) into shared buffer 0 and
  // the registers.  Window cell (ex, ey) is grid cell (bx TW - H + ex, by TH - H + ey), folded.
  CARDIAC_D static void load(const TileArgs<MD>& a, const double* __restrict__ in, int bx, int by,
                             int tx, int ty, double* __restrict__ sm, Patch& st) {
    const int nx = a.g.nx, ny = a.g.ny, pitch = a.g.pitch, bc = a.g.boundary;
    const int gx = bx * TW - H + 2 * tx;
    const int gy0 = by * TH - H + PR * ty;
    const bool vec = VEC && gx >= 0 && gx + 1 < nx;
    // A window reaches at most H cells (plus the ragged part of the last tile) outside the grid: when
    // the grid is larger than that, ONE reflection / wrap maps every index (no integer division —
    // the general fold() was a quarter of all instructions of the kernel, ncu r1 v5).
    const bool once_x = nx > H + TW, once_y = ny > H + TH;
    const int fx0 = once_x ? bidx(gx, nx, bc) : fold(gx, nx, bc);
    const int fx1 = once_x ? bidx(gx + 1, nx, bc) : fold(gx + 1, nx, bc);
    double* s0 = sm + (R + PR * ty) * SP + PADX + 2 * tx;
    // all loads first, then the stores: one exposed memory latency per thread instead of one per row
    double2 v[PR][NV];
#pragma unroll
    for (int k = 0; k < PR; ++k) {
      const int row = (once_y ? bidx(gy0 + k, ny, bc) : fold(gy0 + k, ny, bc)) * pitch;
#pragma unroll
      for (int q = 0; q < NV; ++q) {
        const double* f = in + q * a.g.fstride + row;
        if (vec) {
          v[k][q] = *reinterpret_cast<const double2*>(f + gx);
        } else {
          v[k][q].x = f[fx0];
          v[k][q].y = f[fx1];
        }
      }
    }
#pragma unroll
    for (int k = 0; k < PR; ++k) {
#pragma unroll
      for (int q = 0; q < NV; ++q) {
        if (q < ND) *reinterpret_cast<double2*>(s0 + q * FSZ + k * SP) = v[k][q];
        else { st.g[k][0][q - ND] = v[k][q].x; st.g[k][1][q - ND] = v[k][q].y; }
        if (RK) { st.y[k][0][q] = v[k][q].x; st.y[k][1][q] = v[k][q].y; }
      }
    }
  }

  // Substep S on this thread's patch: reads shared buffer `cur`, writes `nxt` (or, for the last
  // substep, the global output `out`, already offset to the batch member).
  template <int S>
  CARDIAC_D static void stage(const TileArgs<MD>& a, double* __restrict__ out, int bx, int by,
                              int tx, int ty, const double* __restrict__ cur,
                              double* __restrict__ nxt, Patch& st) {
    constexpr int M = R * (S + 1);  // substep S is valid M cells inside the window
    constexpr bool LAST = (S == NS - 1);
    const int ex = 2 * tx, ey = PR * ty;
    if (!(ex + 2 > M && ex < EW - M && ey + PR > M && ey < EH - M)) return;
    const int o = (R + ey) * SP + PADX + ex;
    const double* c = cur + o;

    // rolling window of 2R+1 rows of the own column pair, per diffusing field
    double2 win[ND][2 * R + 1];
    double lw[ND][3], rw[ND][3];  // BOX9 only: columns x-1 and x+2 of rows k-1..k+1
#pragma unroll
    for (int q = 0; q < ND; ++q) {
#pragma unroll
      for (int d = 0; d < 2 * R; ++d) win[q][d + 1] = lds2(c + q * FSZ + (d - R) * SP);
      if (STENCIL == S_BOX9) {
#pragma unroll
        for (int d = 0; d < 2; ++d) {
          lw[q][d + 1] = c[q * FSZ + (d - 1) * SP - 1];
          rw[q][d + 1] = c[q * FSZ + (d - 1) * SP + 2];
        }
      }
    }

#pragma unroll
    for (int k = 0; k < PR; ++k) {
      double s0[ND], s1[ND];
      double2 ctr[ND];
#pragma unroll
      for (int q = 0; q < ND; ++q) {
        const double* ck = c + q * FSZ + k * SP;
#pragma unroll
        for (int d = 0; d < 2 * R; ++d) win[q][d] = win[q][d + 1];
        win[q][2 * R] = lds2(ck + R * SP);
        const double2 w0 = win[q][R];
        ctr[q] = w0;
        if (STENCIL == S_LAP5) {
          const double l = ck[-1], r = ck[2];
          s0[q] = Stencil<S_LAP5>::apply(w0.x, l, w0.y, win[q][0].x, win[q][2].x);
          s1[q] = Stencil<S_LAP5>::apply(w0.y, w0.x, r, win[q][0].y, win[q][2].y);
        } else if (STENCIL == S_LAP9X4) {
          const double2 l = lds2(ck - 2), r = lds2(ck + 2);
          s0[q] = Stencil<S_LAP9X4>::apply(w0.x, l.y, w0.y, win[q][1].x, win[q][3].x, l.x, r.x,
                                           win[q][0].x, win[q][4].x);
          s1[q] = Stencil<S_LAP9X4>::apply(w0.y, w0.x, r.x, win[q][1].y, win[q][3].y, l.y, r.y,
                                           win[q][0].y, win[q][4].y);
        } else {
          lw[q][0] = lw[q][1]; lw[q][1] = lw[q][2]; lw[q][2] = ck[SP - 1];
          rw[q][0] = rw[q][1]; rw[q][1] = rw[q][2]; rw[q][2] = ck[SP + 2];
          s0[q] = Stencil<S_BOX9>::apply(w0.x, lw[q][1], w0.y, win[q][0].x, win[q][2].x, lw[q][0],
                                         win[q][0].y, lw[q][2], win[q][2].y);
          s1[q] = Stencil<S_BOX9>::apply(w0.y, w0.x, rw[q][1], win[q][0].y, win[q][2].y,
                                         win[q][0].x, rw[q][0], win[q][2].x, rw[q][2]);
        }
      }

      double res[2][NV];
#pragma unroll
      for (int h = 0; h < 2; ++h) {
        double z[NV], f[NV];
#pragma unroll
        for (int q = 0; q < NV; ++q)
          z[q] = q < ND ? (h == 0 ? ctr[q < ND ? q : 0].x : ctr[q < ND ? q : 0].y)
                        : st.g[k][h][q >= ND ? q - ND : 0];
        MD::reaction(a.p, z, f);
#pragma unroll
        for (int q = 0; q < ND; ++q) f[q] = fma(a.lapw[q], h == 0 ? s0[q] : s1[q], f[q]);
#pragma unroll
        for (int q = 0; q < NV; ++q) {
          double nv;
          if (!RK) {
            nv = fma(a.a_dt[0], f[q], z[q]);
          } else if (LAST) {
            nv = fma(a.b_dt[S], f[q], S == 0 ? st.y[k][h][q] : st.acc[k][h][q]);
          } else {
            st.acc[k][h][q] = fma(a.b_dt[S], f[q], S == 0 ? st.y[k][h][q] : st.acc[k][h][q]);
            nv = fma(a.a_dt[S], f[q], st.y[k][h][q]);
          }
          res[h][q] = nv;
          if (q >= ND && !LAST) st.g[k][h][q >= ND ? q - ND : 0] = nv;
        }
      }

      if (!LAST) {
#pragma unroll
        for (int q = 0; q < ND; ++q)
          *reinterpret_cast<double2*>(nxt + o + q * FSZ + k * SP) = make_double2(res[0][q], res[1][q]);
      } else {
        // the output tile: window cells at least H inside, clipped to the grid
        const int wy = ey + k;
        const int gx = bx * TW - H + ex, gy = by * TH - H + wy;
        if (wy >= H && wy < EH - H && gy < a.g.ny) {
          double* dst = out + (long long)gy * a.g.pitch + gx;
          if (VEC) {  // H even: a pair is inside the output tile as a whole or not at all
            if (ex >= H && ex < EW - H && gx < a.g.nx) {
              if (gx + 1 < a.g.nx) {
#pragma unroll
                for (int q = 0; q < NV; ++q)
                  *reinterpret_cast<double2*>(dst + q * a.g.fstride) = make_double2(res[0][q], res[1][q]);
              } else {
#pragma unroll
                for (int q = 0; q < NV; ++q) dst[q * a.g.fstride] = res[0][q];
              }
            }
          } else {
#pragma unroll
            for (int h = 0; h < 2; ++h) {
              if (ex + h >= H && ex + h < EW - H && gx + h < a.g.nx) {
#pragma unroll
                for (int q = 0; q < NV; ++q) dst[q * a.g.fstride + h] = res[h][q];
              }
            }
          }
        }
      }
    }
  }

  template <int S>
  CARDIAC_D static void stages_from(const TileArgs<MD>& a, double* __restrict__ out, int bx, int by,
                                    int tx, int ty, double* __restrict__ sm, Patch& st) {
    if constexpr (S < NS) {
      const double* cur = sm + (S & 1) * ND * FSZ;
      double* nxt = sm + ((S + 1) & 1) * ND * FSZ;
      stage<S>(a, out, bx, by, tx, ty, cur, nxt, st);
      if constexpr (S + 1 < NS) {
        __syncthreads();
        stages_from<S + 1>(a, out, bx, by, tx, ty, sm, st);
      }
    }
  }

  // one whole launch worth of substeps on tile (bx, by): in -> out
  CARDIAC_D static void run(const TileArgs<MD>& a, const double* __restrict__ in,
                            double* __restrict__ out, int bx, int by, double* __restrict__ sm) {
    const int tx = threadIdx.x % NTX, ty = threadIdx.x / NTX;
    Patch st;
    load(a, in, bx, by, tx, ty, sm, st);
    __syncthreads();
    stages_from<0>(a, out, bx, by, tx, ty, sm, st);
  }
};

}  // namespace cardiac
