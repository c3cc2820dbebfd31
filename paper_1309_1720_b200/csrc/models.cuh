// models.cuh — device-side pointwise reactions N[z] of the three models (Sect. 2) and the
// smoothed step H_k, shared by every kernel of the CUDA path.
//
// Each model is a struct Model<MODEL, VARIANT> with
//   NV, ND            number of fields / of leading diffusing fields
//   Params            constants derived ON THE HOST from the public parameter block
//                     (reciprocals, products: "explicit methods ... fused multiply-add over division",
//                     PAPER.md:118)
//   derive()          host: public block -> Params
//   reaction()        device: z[NV] -> f[NV] = N[z]
// VARIANT 0 = equations as printed; 1 = PAPER.md:198's tanh(x) -> 2 H_{1/3}(x) - 1 (DESIGN.md f3).
#pragma once
#include <cmath>

#include "fastmath.cuh"

namespace cardiac {

enum { M_FHN = 0, M_KARMA = 1, M_BOCF = 2 };
enum { V_PAPER = 0, V_TANHFREE = 1 };

#define CARDIAC_HD __host__ __device__ __forceinline__

// H_k(x) = t^2 (3 - 2t), t = clamp(k x + 1/2, 0, 1): PAPER.md:94 (its branch form, Q11).
CARDIAC_D double hk(double x, double k) {
  double t = fma(k, x, 0.5);
  t = clamp01(t);
  return t * t * fma(-2.0, t, 3.0);
}

// The models only ever use tanh as (1 +- tanh(a))/2 = 1/(1 + e^{-+2a}) (1 - tanh;
// Eq. 5 and DESIGN.md Q9(v): (1 + tanh)/2).  one_plus_exp<VARIANT>(a) returns q = 1 + e^{-2a}, so
// (1 + tanh a)/2 = 1/q and (1 - tanh a)/2 = (q - 1)/q, and a time constant blended with it,
// 1/(tau1 + dtau/q) = q/(tau1 q + dtau), costs ONE reciprocal instead of two divisions.
// VARIANT 1: tanh(a) -> 2 H_{1/3}(a) - 1, i.e. 1/q = H_{1/3}(a).
CARDIAC_D double ipow(double v, int m) {
  double r = 1.0, b = v;
  while (m > 0) {
    if (m & 1) r *= b;
    b *= b;
    m >>= 1;
  }
  return r;
}

template <int MODEL, int VARIANT>
struct Model;

// ------------------------------------------------------------------ FitzHugh-Nagumo (Eq. 3)
template <int VARIANT>
struct Model<M_FHN, VARIANT> {
  static constexpr int NV = 2, ND = 2, NPARAMS = 5;
  struct Params {
    double D[2];  // D_u, D_v = delta
    double eps, a1, a0;
  };
  static void derive(const double* p, Params& q) {
    q.D[0] = p[0]; q.D[1] = p[1]; q.eps = p[2]; q.a1 = p[3]; q.a0 = p[4];
  }
  CARDIAC_D static void reaction(const Params& q, const double (&z)[NV], double (&f)[NV]) {
    double u = z[0], v = z[1];
    f[0] = fma(-u * u, u, u - v);               // u - v - u^3
    f[1] = q.eps * (fma(-q.a1, v, u) - q.a0);   // eps (u - a1 v - a0)
  }
};

// ------------------------------------------------------------------ Karma (Eq. 4)
template <int VARIANT>
struct Model<M_KARMA, VARIANT> {
  static constexpr int NV = 2, ND = 1, NPARAMS = 9;
  struct Params {
    double D[1];
    double inv_tau_u, inv_tau_v, u_h, u_v, u_star, cR, k;
    int M;
  };
  static void derive(const double* p, Params& q) {
    q.D[0] = p[0]; q.inv_tau_u = 1.0 / p[1]; q.inv_tau_v = 1.0 / p[2];
    q.u_h = p[3]; q.u_v = p[4]; q.u_star = p[5];
    q.cR = 1.0 / (1.0 - std::exp(-p[6]));       // 1/(1 - e^-Re), Q8
    q.M = (int)p[7]; q.k = p[8];
  }
  CARDIAC_D static void reaction(const Params& q, const double (&z)[NV], double (&f)[NV]) {
    double u = z[0], v = z[1];
    // 1 - tanh(a) = 2 e^{-2a}/(1 + e^{-2a}); tanh-free variant: 2 (1 - H_{1/3}(a))
    double omt;
    if (VARIANT == V_TANHFREE) {
      omt = 2.0 * (1.0 - hk(u - q.u_h, 1.0 / 3.0));
    } else {
      double E = exp_c(-2.0 * (u - q.u_h));
      omt = (E + E) * rcp_pos(1.0 + E);
    }
    double vM = (q.M == 6) ? (v * v * v) * (v * v * v) : ipow(v, q.M);
    f[0] = q.inv_tau_u * fma(0.5 * u * u * omt, q.u_star - vM, -u);
    // H_k(x) + H_k(-x) = 1  =>  (cR - v) H - v (1 - H) = cR H - v
    f[1] = q.inv_tau_v * fma(q.cR, hk(u - q.u_v, q.k), -v);
  }
};

// ------------------------------------------------------------------ Bueno-Orovio-Cherry-Fenton (Eq. 5)
template <int VARIANT>
struct Model<M_BOCF, VARIANT> {
  static constexpr int NV = 4, ND = 1, NPARAMS = 30;
  struct Params {
    double D[1];
    double k, u_o, u_u, th_v, th_w, th_vm, th_o;
    double tau_v1m, dtau_vm, inv_tau_vp;
    double tau_w1m, dtau_wm, k_wm, u_wm, inv_tau_wp;
    double inv_tau_fi, tau_o1, dtau_o, tau_so1, dtau_so, k_so, u_so;
    double tau_s1, dtau_s, k_s, u_s, inv_tau_si, inv_tau_winf, winf_star;
    double m2k_wm, m2k_s, m2k_so;  // -2 k: exponent scale of 1 + e^{-2 k (u - u0)}
    int same_o_vm;                 // theta_o == theta_v^- (the epicardial set): H_k(u - theta_o) is H_k(u - theta_v^-)
  };
  static void derive(const double* p, Params& q) {
    q.D[0] = p[0]; q.k = p[1]; q.u_o = p[2]; q.u_u = p[3]; q.th_v = p[4]; q.th_w = p[5];
    q.th_vm = p[6]; q.th_o = p[7];
    q.tau_v1m = p[8]; q.dtau_vm = p[9] - p[8]; q.inv_tau_vp = 1.0 / p[10];
    q.tau_w1m = p[11]; q.dtau_wm = p[12] - p[11]; q.k_wm = p[13]; q.u_wm = p[14];
    q.inv_tau_wp = 1.0 / p[15];
    q.inv_tau_fi = 1.0 / p[16]; q.tau_o1 = p[17]; q.dtau_o = p[18] - p[17];
    q.tau_so1 = p[19]; q.dtau_so = p[20] - p[19]; q.k_so = p[21]; q.u_so = p[22];
    q.tau_s1 = p[23]; q.dtau_s = p[24] - p[23]; q.k_s = p[25]; q.u_s = p[26];
    q.inv_tau_si = 1.0 / p[27]; q.inv_tau_winf = 1.0 / p[28]; q.winf_star = p[29];
    q.m2k_wm = -2.0 * q.k_wm; q.m2k_s = -2.0 * q.k_s; q.m2k_so = -2.0 * q.k_so;
    q.same_o_vm = q.th_o == q.th_vm;
  }

  // gate equations x' = alpha_x(u) x + beta_x(u), x = v, w, s (Q9)
  CARDIAC_D static void gates(const Params& q, double u, double (&alpha)[3], double (&beta)[3]) {
    double h_v = hk(u - q.th_v, q.k), h_w = hk(u - q.th_w, q.k);
    // (uniform branch: with equal thresholds the two are the same instruction sequence on the same input)
    double h_o = hk(u - q.th_o, q.k), h_vm = q.same_o_vm ? h_o : hk(u - q.th_vm, q.k);
    double inv_tau_vm = rcp_pos(fma(h_vm, q.dtau_vm, q.tau_v1m));
    double tau_s = fma(h_w, q.dtau_s, q.tau_s1);
    double inv_tau_wm, inv_tau_s, beta_s;
    if (VARIANT == V_TANHFREE) {
      inv_tau_wm = rcp_pos(fma(q.dtau_wm, hk(q.k_wm * (u - q.u_wm), 1.0 / 3.0), q.tau_w1m));
      inv_tau_s = rcp_pos(tau_s);
      beta_s = hk(q.k_s * (u - q.u_s), 1.0 / 3.0) * inv_tau_s;
    } else {
      // 1/(tau1 + dtau/qw) = qw/(tau1 qw + dtau);  s_inf/tau_s = 1/(qs tau_s), 1/tau_s = qs * that
      double qw = 1.0 + exp_c(q.m2k_wm * (u - q.u_wm));
      inv_tau_wm = qw * rcp_pos(fma(q.tau_w1m, qw, q.dtau_wm));
      double qs = 1.0 + exp_c(q.m2k_s * (u - q.u_s));
      beta_s = rcp_pos(qs * tau_s);
      inv_tau_s = qs * beta_s;
    }
    double v_inf = 1.0 - h_vm;                                      // H_k(theta_v^- - u)
    double w_inf = fma(h_o, q.winf_star, (1.0 - h_o) * fma(-u, q.inv_tau_winf, 1.0));
    double a_v = (1.0 - h_v) * inv_tau_vm, a_w = (1.0 - h_w) * inv_tau_wm;   // H_k(theta - u)/tau^-
    alpha[0] = -fma(h_v, q.inv_tau_vp, a_v);
    beta[0] = a_v * v_inf;
    alpha[1] = -fma(h_w, q.inv_tau_wp, a_w);
    beta[1] = a_w * w_inf;
    alpha[2] = -inv_tau_s;
    beta[2] = beta_s;
  }

  // J_fi + J_so + J_si
  CARDIAC_D static double current(const Params& q, const double (&z)[NV]) {
    double u = z[0], v = z[1], w = z[2], s = z[3];
    double h_v = hk(u - q.th_v, q.k), h_w = hk(u - q.th_w, q.k), h_o = hk(u - q.th_o, q.k);
    double inv_tau_o = rcp_pos(fma(h_o, q.dtau_o, q.tau_o1));
    double inv_tau_so;
    if (VARIANT == V_TANHFREE) {
      inv_tau_so = rcp_pos(fma(q.dtau_so, hk(q.k_so * (u - q.u_so), 1.0 / 3.0), q.tau_so1));
    } else {
      double qso = 1.0 + exp_c(q.m2k_so * (u - q.u_so));
      inv_tau_so = qso * rcp_pos(fma(q.tau_so1, qso, q.dtau_so));
    }
    double J_fi = -v * h_v * (u - q.th_v) * (q.u_u - u) * q.inv_tau_fi;
    double J_so = fma((u - q.u_o) * (1.0 - h_w), inv_tau_o, h_w * inv_tau_so);
    double J_si = -h_w * w * s * q.inv_tau_si;
    return J_fi + J_so + J_si;
  }

  CARDIAC_D static void reaction(const Params& q, const double (&z)[NV], double (&f)[NV]) {
    double alpha[3], beta[3];
    gates(q, z[0], alpha, beta);
    f[0] = -current(q, z);
    f[1] = fma(alpha[0], z[1], beta[0]);
    f[2] = fma(alpha[1], z[2], beta[1]);
    f[3] = fma(alpha[2], z[3], beta[2]);
  }
};

}  // namespace cardiac
