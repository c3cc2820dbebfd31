// fastmath.cuh — branch-free FP64 reciprocal, exp and logistic for the ionic models.
//
// The paper notes that tanh and pow go to the special-function unit with long latency and that
// explicit methods should trade divisions for multiply-adds.  On sm_100a there
// is no FP64 special-function hardware at all: CUDA's exp()/division expand to ~25 / ~12 FP64
// instructions PLUS ~2x as many integer/move instructions (64-bit polynomial coefficients are
// materialised with two 32-bit moves each, the division carries a slow-path call).  ncu on the v1
// kernel showed BOCF issue-bound at 647 warp-instructions per cell-stage of which only 222 were
// FP64 (profiles/r1_v1_cfg4_stage_full.csv).  Measured in round 2: an FP64
// instruction holds a scheduler's issue port for ~2.2 cycles and nothing else issues meanwhile, so
// what a BOCF substep costs is 2.2 x (FP64 instructions) + (all others), and three exponentials and five
// reciprocals were half of its 138 FP64 instructions.  The versions here have no branches and spend
// as few instructions as 1-2 ulp allow:
//   rcp_pos : MUFU.RCP64H seed (rcp.approx.ftz.f64, rel. error e0 <= 2^-23) + ONE third-order step
//             r (1 + e + e^2), e = 1 - b r (remainder e^3 = 2^-69): 3 DFMA                    -> <= 1 ulp
//   exp_c   : x clamped to [-700, 700], n = rint(x 128/ln2) by the 1.5*2^52 trick, two-term Cody-Waite
//             reduction r = x - n ln2/128 (|r| <= 0.0027), e^x = 2^(n>>7) T[n&127] (1 + q),
//             T[j] = 2^(j/128) from a 1 KB table read through L1 (exp_table.inc; a constant-bank table
//             would serialise on the 32 different indices of a warp), q = e^r - 1 = r P4(r) (degree-4
//             Taylor, remainder r^6/720 = 5e-19), result fma(T, q, T): 10 FP64 instructions (the
//             degree-13 polynomial of round 1: 17)                                           -> <= 1.5 ulp
// Neither is correctly rounded; DESIGN.md "Tolerance" budgets 1-2 ulp per operation against the
// oracle's glibc tanh/exp and IEEE division (checked value by value, tests/test_gpu_math.py).
#pragma once

namespace cardiac {

#ifndef CARDIAC_D
#define CARDIAC_D __device__ __forceinline__
#endif

// 2^(j/128), j = 0 .. 127 (global memory, read through L1 with ld.global.nc)
__device__ const double kExp2Tab[128] = {
#include "exp_table.inc"
};

// clamp(t, 0, 1) and clamp(x, -700, 700) decided on the HIGH WORD with integer instructions.
// fmin/fmax on doubles have no single sm_100a instruction: each expands to DSETP (on the FP64 pipe)
// + SEL + FSEL + a NaN-quieting LOP3 + moves (~7 instructions; the BOCF reaction has 14 of them per
// cell, a quarter of its v2 instruction count).  A double with the sign bit set is < 0 (or -0) and a
// non-negative double is >= 1 iff its high word is >= 0x3FF00000, so ONE unsigned compare decides
// "outside [0, 1)"; the replacement value is 0 or 1 by the sign.  Same results as fmin(fmax(t,0),1)
// for every non-NaN t (-0 -> +0); NaN -> 0 or 1 by its sign (a NaN state is already lost).
CARDIAC_D double clamp01(double t) {
  const int hi = __double2hiint(t);
  const bool out = (unsigned)hi >= 0x3FF00000u;
  const int alt = ~(hi >> 31) & 0x3FF00000;   // t < 0 -> 0.0, t >= 1 -> 1.0
  return __hiloint2double(out ? alt : hi, out ? 0 : __double2loint(t));
}
// |x| limited to [0, 700.000123): the magnitude of the HIGH WORD is limited to 0x4085E000 (700.0 =
// 0x4085E000'00000000) with one integer min, the low word is left alone — three integer instructions
// instead of the six of a two-word select (r2: the three exponentials of a BOCF cell paid 36 of the 228
// non-FP64 instructions of a pair-substep for it).  e^x stays finite (overflow is at 709.78), and the
// logistic built on it is at its 0 / 1 limit to 1e-304 long before.
CARDIAC_D double clamp700(double x) {
  const int hi = __double2hiint(x);
  const int m = min(hi & 0x7FFFFFFF, 0x4085E000);
  return __hiloint2double((hi & 0x80000000) | m, __double2loint(x));
}

// b > 0, normal range
CARDIAC_D double rcp_pos(double b) {
  double r;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(b));
  const double e = fma(-b, r, 1.0);
  return fma(r, fma(e, e, e), r);
}

// (literals on purpose: with the coefficients in a __constant__ array ptxas loads them with LDC instead of
// folding them into the DFMAs, measured 2 % slower on the BOCF pair kernels)
CARDIAC_D double exp_c(double x) {
  const double k128L2E = 184.6649652337873;       // 128 log2(e)
  const double kLn2Hi = 0.6931471787393093 / 128.0;       // ln2/128, low 24 mantissa bits zero: n*hi exact
  const double kLn2Lo = 1.8206359985041462e-09 / 128.0;   // ln2/128 - hi (60-digit ln2)
  const double kMagic = 6755399441055744.0;       // 1.5 * 2^52: fma(x, c, magic) rounds x c to an integer
  x = clamp700(x);
  const double t = fma(x, k128L2E, kMagic);
  const int n = __double2loint(t);                // |n| <= 129271
  const double fn = t - kMagic;
  double r = fma(fn, -kLn2Hi, x);
  r = fma(fn, -kLn2Lo, r);
  const double T = __ldg(&kExp2Tab[n & 127]);
  double p = fma(1.0 / 120.0, r, 1.0 / 24.0);     // (e^r - 1)/r = 1 + r/2 + r^2/6 + r^3/24 + r^4/120 (+ r^5/720)
  p = fma(p, r, 1.0 / 6.0);
  p = fma(p, r, 0.5);
  p = fma(p, r, 1.0);
  const double v = fma(T, p * r, T);              // T e^r in [1, 2.01)
  return __hiloint2double(__double2hiint(v) + ((n >> 7) << 20), __double2loint(v));  // v * 2^(n>>7), |n>>7| <= 1010
}

}  // namespace cardiac
