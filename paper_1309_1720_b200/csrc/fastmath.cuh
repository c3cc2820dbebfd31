// fastmath.cuh — branch-free FP64 reciprocal, exp and logistic for the ionic models.
//
// The paper notes that tanh and pow go to the special-function unit with long latency and that
// explicit methods should trade divisions for multiply-adds.  On sm_100a there
// is no FP64 special-function hardware at all: CUDA's exp()/division expand to ~25 / ~12 FP64
// instructions PLUS ~2x as many integer/move instructions (64-bit polynomial coefficients are
// materialised with two 32-bit moves each, the division carries a slow-path call).  ncu on the v1
// kernel showed BOCF issue-bound at 647 warp-instructions per cell-stage of which only 222 were
// FP64 (profiles/r1_v1_cfg4_stage_full.csv).  The versions here keep every coefficient in the
// constant bank (a DFMA operand, no move) and have no branches:
//   rcp_pos : MUFU.RCP64H seed (rcp.approx.ftz.f64, rel. error 2^-23) + two Newton steps -> <= 1 ulp
//   exp_c   : x clamped to [-700, 700], n = rint(x log2 e) by the 1.5*2^52 trick, two-term
//             Cody-Waite reduction, degree-13 Taylor polynomial on |r| <= ln2/2 (remainder 4e-18),
//             2^n added into the exponent field -> <= 1 ulp (+ the clamp: exact 0/1 limits of the
//             logistic are reached to 1e-304)
// Neither is correctly rounded; DESIGN.md "Tolerance" budgets 1 ulp per operation against the
// oracle's glibc tanh/exp and IEEE division.
#pragma once

namespace cardiac {

#ifndef CARDIAC_D
#define CARDIAC_D __device__ __forceinline__
#endif

// 1/k!, k = 13 .. 2 (Horner order), then ln2 split and log2(e)
__constant__ double kExpC[12] = {
    1.0 / 6227020800.0, 1.0 / 479001600.0, 1.0 / 39916800.0, 1.0 / 3628800.0,
    1.0 / 362880.0,     1.0 / 40320.0,     1.0 / 5040.0,     1.0 / 720.0,
    1.0 / 120.0,        1.0 / 24.0,        1.0 / 6.0,        0.5};

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
// |x| >= 700 <=> (high word & 0x7FFFFFFF) >= 0x4085E000 (700.0 = 0x4085E000'00000000)
CARDIAC_D double clamp700(double x) {
  const int hi = __double2hiint(x);
  const bool out = (hi & 0x7FFFFFFF) >= 0x4085E000;
  return __hiloint2double(out ? ((hi & 0x80000000) | 0x4085E000) : hi, out ? 0 : __double2loint(x));
}

// b > 0, normal range
CARDIAC_D double rcp_pos(double b) {
  double r;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(b));
  double e = fma(-b, r, 1.0);
  r = fma(r, e, r);
  e = fma(-b, r, 1.0);
  return fma(r, e, r);
}

CARDIAC_D double exp_c(double x) {
  const double kL2E = 1.4426950408889634074;      // log2(e)
  const double kLn2Hi = 0.6931471787393093;       // ln2 with the low 24 mantissa bits zero: n*hi exact
  const double kLn2Lo = 1.8206359985041462e-09;   // ln2 - kLn2Hi (60-digit ln2)
  const double kMagic = 6755399441055744.0;       // 1.5 * 2^52: fma(x, c, magic) rounds x c to an integer
  x = clamp700(x);
  double t = fma(x, kL2E, kMagic);
  int n = __double2loint(t);
  double fn = t - kMagic;
  double r = fma(fn, -kLn2Hi, x);
  r = fma(fn, -kLn2Lo, r);
  double p = kExpC[0];
#pragma unroll
  for (int i = 1; i < 12; ++i) p = fma(p, r, kExpC[i]);
  p = fma(p, r, 1.0);
  p = fma(p, r, 1.0);   // p = e^r in [0.70, 1.42]
  return __hiloint2double(__double2hiint(p) + (n << 20), __double2loint(p));  // p * 2^n, |n| <= 1010
}

}  // namespace cardiac
