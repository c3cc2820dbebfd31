// stage.cuh — argument blocks and the Laplacian weights shared by all execution plans.
#pragma once
#include "models.cuh"

namespace cardiac {

enum { S_LAP5 = 0, S_LAP9X4 = 1, S_BOX9 = 2 };
enum { B_NOFLUX = 0, B_PERIODIC = 1 };
enum { I_EULER = 0, I_HEUN = 1, I_RK4 = 2, I_RUSH_LARSEN = 3, I_IMPLICIT_EULER = 4 };

// What one stage launch writes (every RK substep is "some combination of local, non-local and
// Euler-like update"):
//   K_SELF : out = in + w_f f(in)                                     Euler; Heun/RK4 stage 1
//   K_BASE : out = w_y y + w_in in + w_f f(in)                         RK4 stages 2,3; Heun stage 2
//   K_RK4F : out = w_y y + w_A A + w_B B + w_in in + w_f f(in)         RK4 stage 4, accumulator-free:
//            y+ = (Y2 + 2 Y3 + Y4 - y)/3 + dt/6 f(Y4)
//   K_RL / K_IE : BOCF, u by Euler, gates by Rush-Larsen / implicit Euler
enum { K_SELF = 0, K_BASE = 1, K_RK4F = 2, K_RL = 3, K_IE = 4 };

__host__ __device__ constexpr int stencil_radius(int stencil) { return stencil == S_LAP9X4 ? 2 : 1; }
// lap(U) = lap_norm * (integer-weight stencil sum) / dx^2
__host__ __device__ constexpr double stencil_norm(int stencil) {
  return stencil == S_LAP9X4 ? 1.0 / 12.0 : (stencil == S_BOX9 ? 1.0 / 6.0 : 1.0);
}

// State buffers are [batch][n_v][ny] rows of `pitch` doubles (pitch >= nx, multiple of 16 so every
// row starts 128-byte aligned); x fastest.
struct Geom {
  int nx, ny, pitch, boundary;
  long long fstride;  // doubles between fields  (= pitch * ny * nz)
  long long bstride;  // doubles between batch members (= fstride * n_v)
  int nz;             // 1: the paper's 2-D problem; > 1: 3-D, planes of pitch * ny doubles
  int zstride;        // doubles between planes (= pitch * ny)
};

template <class MD>
struct StageArgs {
  const double* in;  // stage input (read with halo for the diffusing fields)
  const double* y;   // state at the start of the step (pointwise)
  const double* A;   // Y2 (pointwise, K_RK4F)
  const double* B;   // Y3 (pointwise, K_RK4F)
  double* out;       // may alias y (in-place final stage), never in
  Geom g;
  double w_y, w_in, w_A, w_B, w_f;  // w_f already contains dt
  double dt;
  double lapw[MD::ND];  // D_f * stencil_norm / dx^2
  typename MD::Params p;
};

// out-of-range index -> in-range index ("flip displacement vectors which cross the
// domain boundary back into the domain"; index reflection about the boundary node, Q3;
// periodic: "mapping to the opposite-edge values")
CARDIAC_D int bidx(int i, int n, int boundary) {
  if (boundary == B_PERIODIC) return i < 0 ? i + n : (i >= n ? i - n : i);
  return i < 0 ? -i : (i >= n ? 2 * (n - 1) - i : i);
}

// integer-weight stencil sums
template <int STENCIL>
struct Stencil;
template <>
struct Stencil<S_LAP5> {
  // c, then W, E, S, N
  CARDIAC_D static double apply(double c, double w, double e, double s, double n) {
    return fma(-4.0, c, (w + e) + (s + n));
  }
};
template <>
struct Stencil<S_LAP9X4> {
  CARDIAC_D static double apply(double c, double w1, double e1, double s1, double n1, double w2,
                                double e2, double s2, double n2) {
    double a1 = (w1 + e1) + (s1 + n1), a2 = (w2 + e2) + (s2 + n2);
    return fma(-60.0, c, fma(16.0, a1, -a2));
  }
};
template <>
struct Stencil<S_BOX9> {
  CARDIAC_D static double apply(double c, double w, double e, double s, double n, double sw,
                                double se, double nw, double ne) {
    double ax = (w + e) + (s + n), dg = (sw + se) + (nw + ne);
    return fma(-20.0, c, fma(4.0, ax, dg));
  }
};

// 128-bit accesses of an x-adjacent pair of cells ("vector width 2 for doubles")
CARDIAC_D double2 ld2(const double* p) { return *reinterpret_cast<const double2*>(p); }
CARDIAC_D void prefetch_l1(const double* p) { asm volatile("prefetch.global.L1 [%0];" ::"l"(p)); }
CARDIAC_D void st2(double* p, double a, double b) { *reinterpret_cast<double2*>(p) = make_double2(a, b); }

// integer-weight stencil sums of the two cells (x, x+1) of row `row`; interior, no boundary logic
template <int STENCIL>
CARDIAC_D void stencil_pair(const double* __restrict__ U, int row, int x, int pitch, double2 c,
                            double& s0, double& s1) {
  const double* p = U + row + x;
  if (STENCIL == S_LAP5) {
    const double w = p[-1], e = p[2];
    const double2 s = ld2(p - pitch), n = ld2(p + pitch);
    s0 = Stencil<S_LAP5>::apply(c.x, w, c.y, s.x, n.x);
    s1 = Stencil<S_LAP5>::apply(c.y, c.x, e, s.y, n.y);
  } else if (STENCIL == S_LAP9X4) {
    const double2 l = ld2(p - 2), r = ld2(p + 2);
    const double2 a1 = ld2(p - pitch), b1 = ld2(p + pitch);
    const double2 a2 = ld2(p - 2 * pitch), b2 = ld2(p + 2 * pitch);
    s0 = Stencil<S_LAP9X4>::apply(c.x, l.y, c.y, a1.x, b1.x, l.x, r.x, a2.x, b2.x);
    s1 = Stencil<S_LAP9X4>::apply(c.y, c.x, r.x, a1.y, b1.y, l.y, r.y, a2.y, b2.y);
  } else {
    const double w = p[-1], e = p[2];
    const double2 s = ld2(p - pitch), n = ld2(p + pitch);
    const double sw = p[-pitch - 1], se = p[-pitch + 2], nw = p[pitch - 1], ne = p[pitch + 2];
    s0 = Stencil<S_BOX9>::apply(c.x, w, c.y, s.x, n.x, sw, s.y, nw, n.y);
    s1 = Stencil<S_BOX9>::apply(c.y, c.x, e, s.y, n.y, s.x, se, n.x, ne);
  }
}

// ... of ONE interior cell at offset o of the field: the operands in the same Stencil<>::apply positions as either
// half of stencil_pair (c, W, E, S, N, then the second ring) — the same bits
template <int STENCIL>
CARDIAC_D double stencil_cell(const double* __restrict__ U, int o, int pitch, double c) {
  const double* p = U + o;
  if (STENCIL == S_LAP5) {
    return Stencil<S_LAP5>::apply(c, p[-1], p[1], p[-pitch], p[pitch]);
  } else if (STENCIL == S_LAP9X4) {
    return Stencil<S_LAP9X4>::apply(c, p[-1], p[1], p[-pitch], p[pitch], p[-2], p[2], p[-2 * pitch], p[2 * pitch]);
  } else {
    return Stencil<S_BOX9>::apply(c, p[-1], p[1], p[-pitch], p[pitch], p[-pitch - 1], p[-pitch + 1], p[pitch - 1],
                                  p[pitch + 1]);
  }
}

// one cell with the boundary rule applied per axis (Q3)
template <int STENCIL>
CARDIAC_D double stencil_edge(const double* __restrict__ U, int i, int j, int nx, int ny, int pitch,
                              int bc, double c) {
  const int rw1 = bidx(i - 1, nx, bc), re1 = bidx(i + 1, nx, bc);
  const int row = j * pitch;
  const int rs1 = bidx(j - 1, ny, bc) * pitch, rn1 = bidx(j + 1, ny, bc) * pitch;
  if (STENCIL == S_LAP5) {
    return Stencil<S_LAP5>::apply(c, U[row + rw1], U[row + re1], U[rs1 + i], U[rn1 + i]);
  } else if (STENCIL == S_LAP9X4) {
    const int rw2 = bidx(i - 2, nx, bc), re2 = bidx(i + 2, nx, bc);
    const int rs2 = bidx(j - 2, ny, bc) * pitch, rn2 = bidx(j + 2, ny, bc) * pitch;
    return Stencil<S_LAP9X4>::apply(c, U[row + rw1], U[row + re1], U[rs1 + i], U[rn1 + i],
                                    U[row + rw2], U[row + re2], U[rs2 + i], U[rn2 + i]);
  } else {
    return Stencil<S_BOX9>::apply(c, U[row + rw1], U[row + re1], U[rs1 + i], U[rn1 + i],
                                  U[rs1 + rw1], U[rs1 + re1], U[rn1 + rw1], U[rn1 + re1]);
  }
}

// ... of a pair (x, x+1) INSIDE the grid whose stencil may reach across the boundary: the pair's vertical
// neighbours stay 128-bit loads from the reflected / wrapped ROW; only the four (six) horizontal
// neighbour values are single loads through the boundary rule.  Same operands in the same
// Stencil<>::apply positions as stencil_pair: the same bits.  U points at the field (plane), x is even.
template <int STENCIL>
CARDIAC_D void stencil_pair_bc(const double* __restrict__ U, int x, int j, int nx, int ny, int pitch, int bc,
                               double2 c, double& s0, double& s1) {
  const int row = j * pitch;
  const int xw1 = bidx(x - 1, nx, bc), xe1 = bidx(x + 2, nx, bc);
  const int rs1 = bidx(j - 1, ny, bc) * pitch, rn1 = bidx(j + 1, ny, bc) * pitch;
  const double w1 = U[row + xw1], e1 = U[row + xe1];
  const double2 s = ld2(U + rs1 + x), n = ld2(U + rn1 + x);
  if (STENCIL == S_LAP5) {
    s0 = Stencil<S_LAP5>::apply(c.x, w1, c.y, s.x, n.x);
    s1 = Stencil<S_LAP5>::apply(c.y, c.x, e1, s.y, n.y);
  } else if (STENCIL == S_LAP9X4) {
    const double w2 = U[row + bidx(x - 2, nx, bc)], e2 = U[row + bidx(x + 3, nx, bc)];
    const double2 a2 = ld2(U + bidx(j - 2, ny, bc) * pitch + x), b2 = ld2(U + bidx(j + 2, ny, bc) * pitch + x);
    s0 = Stencil<S_LAP9X4>::apply(c.x, w1, c.y, s.x, n.x, w2, e1, a2.x, b2.x);
    s1 = Stencil<S_LAP9X4>::apply(c.y, c.x, e1, s.y, n.y, w1, e2, a2.y, b2.y);
  } else {
    const double sw = U[rs1 + xw1], se = U[rs1 + xe1], nw = U[rn1 + xw1], ne = U[rn1 + xe1];
    s0 = Stencil<S_BOX9>::apply(c.x, w1, c.y, s.x, n.x, sw, s.y, nw, n.y);
    s1 = Stencil<S_BOX9>::apply(c.y, c.x, e1, s.y, n.y, s.x, se, n.x, ne);
  }
}

// 3-D: what the z axis adds to the integer-weight sum of the 2-D stencil of the same family
// (7-point = LAP5 + z arm, 13-point = LAP9X4 + z arm; same per-axis weights, DESIGN.md f4)
template <int STENCIL>
struct StencilZ;
template <>
struct StencilZ<S_LAP5> {
  CARDIAC_D static double apply(double c, double d1, double u1) { return fma(-2.0, c, d1 + u1); }
};
template <>
struct StencilZ<S_LAP9X4> {
  CARDIAC_D static double apply(double c, double d1, double u1, double d2, double u2) {
    return fma(-30.0, c, fma(16.0, d1 + u1, -(d2 + u2)));
  }
};

// the RK combination of one field value, shared by every plan
template <int KIND>
CARDIAC_D double combine(double w_y, double w_in, double w_A, double w_B, double w_f, double y,
                         double in, double A, double B, double f) {
  if (KIND == K_SELF) return fma(w_f, f, in);
  if (KIND == K_BASE) return fma(w_f, f, fma(w_in, in, w_y * y));
  return fma(w_f, f, fma(w_in, in, fma(w_B, B, fma(w_A, A, w_y * y))));
}

}  // namespace cardiac
