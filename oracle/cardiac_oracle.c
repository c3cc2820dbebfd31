/*
 * cardiac_oracle.c — TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, obviously-correct CPU restatement (FP64, one thread unless built with -fopenmp,
 * which only splits independent row loops and changes no arithmetic) of what the hot path
 * computes: the explicit time step of  dz/dt = D lap(z) + N[z]  (Eq. 1) with no-flux
 * boundaries (PAPER.md:41 Eq. 2, :104 Fig. 1, :114) for the three models of PAPER.md Sect. 2 and
 * the integrators of PAPER.md:116-118.  There is no closed form for the nonlinear result, so the
 * oracle IS the algorithm, step by step, in the paper's order ("the nonlocal terms
 * ... are computed first, followed by the calculation of the local terms, after which the results
 * are combined and used to update each field"), with separate arrays per stage and no fusion,
 * blocking or reordering.  Readings of the paper where it is silent or garbled are listed in
 * DESIGN.md (Q1..Q16) and cited below.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * call this.  It shares no code, header, table or constant generator with the CUDA path
 * (paper_1309_1720_b200/csrc); the constants below are typed from the paper / DESIGN.md on their own.
 *
 * Parity build: gcc -O2 -ffp-contract=off (no FMA contraction).  Pins: tests/test_oracle_*.py
 * (-m "not gpu").  Unpinned: nothing on the hot path; long chaotic runs are "parity unpinned"
 * by nature and are not compared.
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>

#ifdef _OPENMP
#define OMP_FOR _Pragma("omp parallel for")
#else
#define OMP_FOR
#endif

enum { M_FHN = 0, M_KARMA = 1, M_BOCF = 2 };
enum { S_LAP5 = 0, S_LAP9X4 = 1, S_BOX9 = 2 };
enum { I_EULER = 0, I_HEUN = 1, I_RK4 = 2, I_RUSH_LARSEN = 3, I_IMPLICIT_EULER = 4 };
enum { B_NOFLUX = 0, B_PERIODIC = 1 };
enum { V_PAPER = 0, V_TANHFREE = 1 };

/* ------------------------------------------------------------------ model tables */

int oracle_num_fields(int model) {
  switch (model) { case M_FHN: return 2; case M_KARMA: return 2; case M_BOCF: return 4; }
  return -1;
}

int oracle_num_params(int model) {
  switch (model) { case M_FHN: return 5; case M_KARMA: return 9; case M_BOCF: return 30; }
  return -1;
}

/* number of leading fields that diffuse: FHN u and v, Karma u,
 * BOCF u.  DESIGN.md Q5. */
static int num_diffusing(int model) { return model == M_FHN ? 2 : 1; }

/* Parameter blocks (same order as include/cardiac.h documents for the product, typed here
 * independently). */
int oracle_default_params(int model, double* p) {
  if (model == M_FHN) {
    /* (delta, eps, a1, a0) = (1.5, 0.05, 1.5, -0.1); the u-equation has unit diffusion */
    p[0] = 1.0;   /* D_u */
    p[1] = 1.5;   /* delta = D_v */
    p[2] = 0.05;  /* epsilon */
    p[3] = 1.5;   /* a1 */
    p[4] = -0.1;  /* a0 */
    return 0;
  }
  if (model == M_KARMA) {
    /* (Re, M, gamma) = (1.0, 6, 0.0011); the rest "from Ref. [2]" — recalled values,
     * DESIGN.md Q7; H_k with k = 28.4 */
    p[0] = 0.0011; /* gamma, cm^2/ms */
    p[1] = 2.5;    /* tau_u, ms */
    p[2] = 250.0;  /* tau_v, ms */
    p[3] = 3.0;    /* u_h */
    p[4] = 1.0;    /* u_v */
    p[5] = 1.5415; /* u_star */
    p[6] = 1.0;    /* Re */
    p[7] = 6.0;    /* M */
    p[8] = 28.4;   /* k */
    return 0;
  }
  if (model == M_BOCF) {
    /* D = 1.171 cm^2/s = 1.171e-3 cm^2/ms (time constants are in ms, Q9(ii));
     * epicardial set of Ref. [3] — recalled values, Q9(i); k = 28.4 */
    p[0] = 1.171e-3; /* D */
    p[1] = 28.4;     /* k */
    p[2] = 0.0;      /* u_o */
    p[3] = 1.55;     /* u_u */
    p[4] = 0.3;      /* theta_v */
    p[5] = 0.13;     /* theta_w */
    p[6] = 0.006;    /* theta_v_minus */
    p[7] = 0.006;    /* theta_o */
    p[8] = 60.0;     /* tau_v1_minus */
    p[9] = 1150.0;   /* tau_v2_minus */
    p[10] = 1.4506;  /* tau_v_plus */
    p[11] = 60.0;    /* tau_w1_minus */
    p[12] = 15.0;    /* tau_w2_minus */
    p[13] = 65.0;    /* k_w_minus */
    p[14] = 0.03;    /* u_w_minus */
    p[15] = 200.0;   /* tau_w_plus */
    p[16] = 0.11;    /* tau_fi */
    p[17] = 400.0;   /* tau_o1 */
    p[18] = 6.0;     /* tau_o2 */
    p[19] = 30.0181; /* tau_so1 */
    p[20] = 0.9957;  /* tau_so2 */
    p[21] = 2.0458;  /* k_so */
    p[22] = 0.65;    /* u_so */
    p[23] = 2.7342;  /* tau_s1 */
    p[24] = 16.0;    /* tau_s2 */
    p[25] = 2.0994;  /* k_s */
    p[26] = 0.9087;  /* u_s */
    p[27] = 1.8875;  /* tau_si */
    p[28] = 0.07;    /* tau_w_inf */
    p[29] = 0.94;    /* w_inf_star */
    return 0;
  }
  return -1;
}

/* ------------------------------------------------------------------ H_k */

/* Smoothed step with cubic interpolation, written in the paper's branch form:
 *   0 for kx < -0.5;  (3 - 2kx - 1)(kx + 0.5)^2 for -0.5 <= kx <= 0.5;  1 for kx > 0.5. */
double oracle_hk(double x, double k) {
  double kx = k * x;
  if (kx < -0.5) return 0.0;
  if (kx > 0.5) return 1.0;
  return (3.0 - 2.0 * kx - 1.0) * (kx + 0.5) * (kx + 0.5);
}

/* tanh of the printed equations, or its PAPER.md:198 replacement 2 H_k'(x) - 1 with k' = 1/3, the
 * value that matches the slope of tanh at 0 (d/dx 2H_k'(x) = 3k'; DESIGN.md f3). */
static double tanh_v(double x, int variant) {
  if (variant == V_TANHFREE) return 2.0 * oracle_hk(x, 1.0 / 3.0) - 1.0;
  return tanh(x);
}

/* ------------------------------------------------------------------ reactions N[z], pointwise */

/* PAPER.md:48-51, Eq. 3 */
static void reaction_fhn(const double* p, const double* z, double* f) {
  double eps = p[2], a1 = p[3], a0 = p[4];
  double u = z[0], v = z[1];
  f[0] = u - v - u * u * u;
  f[1] = eps * (u - a1 * v - a0);
}

/* PAPER.md:58-60, Eq. 4 */
static void reaction_karma(const double* p, const double* z, double* f, int variant) {
  double tau_u = p[1], tau_v = p[2], u_h = p[3], u_v = p[4], u_star = p[5], Re = p[6], M = p[7],
         k = p[8];
  double u = z[0], v = z[1];
  f[0] = ((u * u / 2.0) * (1.0 - tanh_v(u - u_h, variant)) * (u_star - pow(v, M)) - u) / tau_u;
  f[1] = ((1.0 / (1.0 - exp(-Re)) - v) * oracle_hk(u - u_v, k) - v * oracle_hk(u_v - u, k)) / tau_v;
}

/* BOCF gate coefficients: d x/dt = alpha_x(u) x + beta_x(u) for x = v, w, s.
 * PAPER.md:86-88 for v and w; the s equation of Eq. 5 is of the same form with
 * alpha_s = -1/tau_s(u), beta_s = s_inf(u)/tau_s(u) (division: DESIGN.md Q9(iii)).
 * Undefined symbols of the paper follow DESIGN.md Q9(v),(vi). */
static void bocf_gates(const double* p, double u, int variant, double* alpha, double* beta) {
  double k = p[1];
  double theta_v = p[4], theta_w = p[5], theta_vm = p[6], theta_o = p[7];
  double tau_v1m = p[8], tau_v2m = p[9], tau_vp = p[10];
  double tau_w1m = p[11], tau_w2m = p[12], k_wm = p[13], u_wm = p[14], tau_wp = p[15];
  double tau_s1 = p[23], tau_s2 = p[24], k_s = p[25], u_s = p[26];
  double tau_winf = p[28], winf_star = p[29];

  double tau_vm = tau_v1m + oracle_hk(u - theta_vm, k) * (tau_v2m - tau_v1m);
  double tau_wm = tau_w1m + (tau_w2m - tau_w1m) * (1.0 + tanh_v(k_wm * (u - u_wm), variant)) / 2.0;
  double tau_s = tau_s1 + oracle_hk(u - theta_w, k) * (tau_s2 - tau_s1);
  double v_inf = oracle_hk(theta_vm - u, k);
  double w_inf = (1.0 - oracle_hk(u - theta_o, k)) * (1.0 - u / tau_winf)
               + oracle_hk(u - theta_o, k) * winf_star;
  double s_inf = (1.0 + tanh_v(k_s * (u - u_s), variant)) / 2.0;

  alpha[0] = -oracle_hk(u - theta_v, k) / tau_vp - oracle_hk(theta_v - u, k) / tau_vm;
  beta[0] = oracle_hk(theta_v - u, k) * v_inf / tau_vm;
  alpha[1] = -oracle_hk(u - theta_w, k) / tau_wp - oracle_hk(theta_w - u, k) / tau_wm;
  beta[1] = oracle_hk(theta_w - u, k) * w_inf / tau_wm;
  alpha[2] = -1.0 / tau_s;
  beta[2] = s_inf / tau_s;
}

/* total ionic current J_fi + J_so + J_si */
static double bocf_current(const double* p, const double* z, int variant) {
  double k = p[1];
  double u_o = p[2], u_u = p[3], theta_v = p[4], theta_w = p[5], theta_o = p[7];
  double tau_fi = p[16], tau_o1 = p[17], tau_o2 = p[18];
  double tau_so1 = p[19], tau_so2 = p[20], k_so = p[21], u_so = p[22], tau_si = p[27];
  double u = z[0], v = z[1], w = z[2], s = z[3];

  double tau_o = tau_o1 + oracle_hk(u - theta_o, k) * (tau_o2 - tau_o1);
  double tau_so = tau_so1 + (tau_so2 - tau_so1) * (1.0 + tanh_v(k_so * (u - u_so), variant)) / 2.0;

  double J_fi = -v * oracle_hk(u - theta_v, k) * (u - theta_v) * (u_u - u) / tau_fi;
  double J_so = (u - u_o) * oracle_hk(theta_w - u, k) / tau_o + oracle_hk(u - theta_w, k) / tau_so;
  double J_si = -oracle_hk(u - theta_w, k) * w * s / tau_si;
  return J_fi + J_so + J_si;
}

/* PAPER.md:67-73, Eq. 5 */
static void reaction_bocf(const double* p, const double* z, double* f, int variant) {
  double alpha[3], beta[3];
  bocf_gates(p, z[0], variant, alpha, beta);
  f[0] = -bocf_current(p, z, variant);
  f[1] = alpha[0] * z[1] + beta[0];
  f[2] = alpha[1] * z[2] + beta[1];
  f[3] = alpha[2] * z[3] + beta[2];
}

/* N[z] at one cell: z[n_v] -> f[n_v]. */
int oracle_reaction(int model, int variant, const double* p, const double* z, double* f) {
  switch (model) {
    case M_FHN: reaction_fhn(p, z, f); return 0;
    case M_KARMA: reaction_karma(p, z, f, variant); return 0;
    case M_BOCF: reaction_bocf(p, z, f, variant); return 0;
  }
  return -1;
}

/* ------------------------------------------------------------------ Laplacian + boundary */

/* No-flux: reflect an out-of-range index about the boundary node, -m -> m, N-1+m -> N-1-m
 * (PAPER.md:104 Fig. 1 "mirroring", :114; Q3).  Periodic: wrap. */
static int bidx(int idx, int n, int boundary) {
  if (boundary == B_PERIODIC) return ((idx % n) + n) % n;
  if (idx < 0) return -idx;
  if (idx > n - 1) return 2 * (n - 1) - idx;
  return idx;
}

/* L = lap(U) on an ny x nx grid (x fastest), spacing dx = dy (Q2), in difference form
 * sum_m c_m [(U_{+m} - U_0) + (U_{-m} - U_0)] so that a uniform field gives exactly 0. */
int oracle_laplacian(const double* U, double* L, int nx, int ny, double dx, int stencil, int boundary) {
  int r = (stencil == S_LAP9X4) ? 2 : 1;
  if (stencil < 0 || stencil > 2 || nx < 2 * r + 1 || ny < 2 * r + 1) return -1;
  double h2 = dx * dx;
#ifdef _OPENMP
#pragma omp parallel for
#endif
  for (int j = 0; j < ny; ++j) {
    for (int i = 0; i < nx; ++i) {
#define UU(di, dj) U[(size_t)bidx(j + (dj), ny, boundary) * nx + bidx(i + (di), nx, boundary)]
      double u0 = U[(size_t)j * nx + i];
      double s;
      if (stencil == S_LAP5) {
        /* Eq. 6 with alpha_a = 1, alpha_d = 0 (Q1) */
        s = ((UU(1, 0) - u0) + (UU(-1, 0) - u0)) + ((UU(0, 1) - u0) + (UU(0, -1) - u0));
      } else if (stencil == S_LAP9X4) {
        /* per axis (-1/12, 4/3, -5/2, 4/3, -1/12) (Q4) */
        double c1 = 4.0 / 3.0, c2 = -1.0 / 12.0;
        double ax = c1 * ((UU(1, 0) - u0) + (UU(-1, 0) - u0)) + c2 * ((UU(2, 0) - u0) + (UU(-2, 0) - u0));
        double ay = c1 * ((UU(0, 1) - u0) + (UU(0, -1) - u0)) + c2 * ((UU(0, 2) - u0) + (UU(0, -2) - u0));
        s = ax + ay;
      } else {
        /* Eq. 6 with alpha_a = 2/3, alpha_d = 1/6 (Q1) */
        double aa = 2.0 / 3.0, ad = 1.0 / 6.0;
        double axial = ((UU(1, 0) - u0) + (UU(-1, 0) - u0)) + ((UU(0, 1) - u0) + (UU(0, -1) - u0));
        double diag = ((UU(1, 1) - u0) + (UU(-1, -1) - u0)) + ((UU(1, -1) - u0) + (UU(-1, 1) - u0));
        s = aa * axial + ad * diag;
      }
#undef UU
      L[(size_t)j * nx + i] = s / h2;
    }
  }
  return 0;
}

/* 3-D ("three-dimensional simulations (corresponding to ventricular tissue)"; DESIGN.md f4):
 * L = lap(U) on an nz x ny x nx grid (x fastest), spacing dx = dy = dz, the same per-axis weights
 * as in 2-D applied along x, y and z — S_LAP5 becomes the 7-point stencil, S_LAP9X4 the 13-point
 * 4th-order cross; Eq. 6's 3 x 3 box (S_BOX9) has no 3-D counterpart in the paper: rejected.
 * Same index reflection / wrap per axis, same difference form. */
int oracle_laplacian3d(const double* U, double* L, int nx, int ny, int nz, double dx, int stencil,
                       int boundary) {
  int r = (stencil == S_LAP9X4) ? 2 : 1;
  if ((stencil != S_LAP5 && stencil != S_LAP9X4) || nx < 2 * r + 1 || ny < 2 * r + 1 || nz < 2 * r + 1)
    return -1;
  double h2 = dx * dx;
#ifdef _OPENMP
#pragma omp parallel for
#endif
  for (int k = 0; k < nz; ++k) {
    for (int j = 0; j < ny; ++j) {
      for (int i = 0; i < nx; ++i) {
#define UU(di, dj, dk)                                                                   \
  U[((size_t)bidx(k + (dk), nz, boundary) * ny + bidx(j + (dj), ny, boundary)) * nx + \
    bidx(i + (di), nx, boundary)]
        double u0 = U[((size_t)k * ny + j) * nx + i];
        double s;
        if (stencil == S_LAP5) {
          double ax = (UU(1, 0, 0) - u0) + (UU(-1, 0, 0) - u0);
          double ay = (UU(0, 1, 0) - u0) + (UU(0, -1, 0) - u0);
          double az = (UU(0, 0, 1) - u0) + (UU(0, 0, -1) - u0);
          s = (ax + ay) + az;
        } else {
          double c1 = 4.0 / 3.0, c2 = -1.0 / 12.0;
          double ax = c1 * ((UU(1, 0, 0) - u0) + (UU(-1, 0, 0) - u0)) + c2 * ((UU(2, 0, 0) - u0) + (UU(-2, 0, 0) - u0));
          double ay = c1 * ((UU(0, 1, 0) - u0) + (UU(0, -1, 0) - u0)) + c2 * ((UU(0, 2, 0) - u0) + (UU(0, -2, 0) - u0));
          double az = c1 * ((UU(0, 0, 1) - u0) + (UU(0, 0, -1) - u0)) + c2 * ((UU(0, 0, 2) - u0) + (UU(0, 0, -2) - u0));
          s = (ax + ay) + az;
        }
#undef UU
        L[((size_t)k * ny + j) * nx + i] = s / h2;
      }
    }
  }
  return 0;
}

/* ------------------------------------------------------------------ right-hand side */

typedef struct {
  int model, stencil, integrator, boundary, variant;
  int nx, ny, nz, nv, nd;   /* nz == 1: the 2-D problem of the paper */
  double dx, dt;
  const double* p;
} problem;

/* F = D lap(Z) + N[Z] for one state Z[n_v][nz][ny][nx]; lapbuf is scratch of nz*ny*nx doubles.
 * Order as in PAPER.md:132: non-local terms first, then the local terms, then combined. */
static void rhs(const problem* q, const double* Z, double* F, double* lapbuf) {
  size_t n = (size_t)q->nx * q->ny * q->nz;
  for (int f = 0; f < q->nd; ++f) {
    double D = (q->model == M_FHN) ? q->p[f] : q->p[0];
    if (q->nz > 1)
      oracle_laplacian3d(Z + f * n, lapbuf, q->nx, q->ny, q->nz, q->dx, q->stencil, q->boundary);
    else
      oracle_laplacian(Z + f * n, lapbuf, q->nx, q->ny, q->dx, q->stencil, q->boundary);
#ifdef _OPENMP
#pragma omp parallel for
#endif
    for (long c = 0; c < (long)n; ++c) F[f * n + c] = D * lapbuf[c];
  }
  for (int f = q->nd; f < q->nv; ++f)
    for (size_t c = 0; c < n; ++c) F[f * n + c] = 0.0;
#ifdef _OPENMP
#pragma omp parallel for
#endif
  for (long c = 0; c < (long)n; ++c) {
    double z[4], g[4];
    for (int f = 0; f < q->nv; ++f) z[f] = Z[f * n + c];
    oracle_reaction(q->model, q->variant, q->p, z, g);
    for (int f = 0; f < q->nv; ++f) F[f * n + c] = F[f * n + c] + g[f];
  }
}

int oracle_rhs(int model, int nx, int ny, double dx, int scheme, const double* params,
               const double* Z, double* F) {
  double pdef[32];
  problem q;
  q.model = model; q.stencil = scheme & 0xff; q.integrator = (scheme >> 8) & 0xff;
  q.boundary = (scheme >> 16) & 0xff; q.variant = (scheme >> 24) & 0xff;
  q.nx = nx; q.ny = ny; q.nz = 1; q.dx = dx; q.dt = 0.0;
  q.nv = oracle_num_fields(model);
  if (q.nv < 0) return -1;
  q.nd = num_diffusing(model);
  if (params) q.p = params; else { oracle_default_params(model, pdef); q.p = pdef; }
  double* lapbuf = (double*)malloc(sizeof(double) * nx * ny);
  if (!lapbuf) return -2;
  rhs(&q, Z, F, lapbuf);
  free(lapbuf);
  return 0;
}

/* ------------------------------------------------------------------ integrators */

/* One time step of one state, in place.  w = workspace of 5*n_v*n + n doubles. */
static void step_once(const problem* q, double* Z, double* w) {
  size_t n = (size_t)q->nx * q->ny * q->nz, N = n * q->nv;
  double dt = q->dt;
  double *K1 = w, *K2 = w + N, *K3 = w + 2 * N, *K4 = w + 3 * N, *Y = w + 4 * N, *lapbuf = w + 5 * N;

  if (q->integrator == I_EULER) {
    /* PAPER.md:118; z+ = z + dt f(z) */
    rhs(q, Z, K1, lapbuf);
    OMP_FOR
    for (long c = 0; c < (long)N; ++c) Z[c] = Z[c] + dt * K1[c];
  } else if (q->integrator == I_HEUN) {
    /* PAPER.md:118, :132, Fig. 2; explicit trapezoid (Q12) */
    rhs(q, Z, K1, lapbuf);
    OMP_FOR
    for (long c = 0; c < (long)N; ++c) Y[c] = Z[c] + dt * K1[c];
    rhs(q, Y, K2, lapbuf);
    OMP_FOR
    for (long c = 0; c < (long)N; ++c) Z[c] = Z[c] + (dt / 2.0) * (K1[c] + K2[c]);
  } else if (q->integrator == I_RK4) {
    /* PAPER.md:118 "classic Runge-Kutta" */
    rhs(q, Z, K1, lapbuf);
    OMP_FOR
    for (long c = 0; c < (long)N; ++c) Y[c] = Z[c] + (dt / 2.0) * K1[c];
    rhs(q, Y, K2, lapbuf);
    OMP_FOR
    for (long c = 0; c < (long)N; ++c) Y[c] = Z[c] + (dt / 2.0) * K2[c];
    rhs(q, Y, K3, lapbuf);
    OMP_FOR
    for (long c = 0; c < (long)N; ++c) Y[c] = Z[c] + dt * K3[c];
    rhs(q, Y, K4, lapbuf);
    OMP_FOR
    for (long c = 0; c < (long)N; ++c)
      Z[c] = Z[c] + (dt / 6.0) * (K1[c] + 2.0 * K2[c] + 2.0 * K3[c] + K4[c]);
  } else {
    /* BOCF only: u by explicit Euler; the non-diffusive variables
     * x' = alpha_x(u) x + beta_x(u), coefficients frozen at u^n, by
     *   Rush-Larsen:    x+ = x e^{alpha dt} + (beta/alpha)(e^{alpha dt} - 1)   (exponential time differencing)
     *   implicit Euler: x+ = (x + dt beta) / (1 - dt alpha). */
    rhs(q, Z, K1, lapbuf); /* only the u component is used */
    OMP_FOR
    for (long c = 0; c < (long)n; ++c) {
      double alpha[3], beta[3];
      double u = Z[c];
      bocf_gates(q->p, u, q->variant, alpha, beta);
      for (int g = 0; g < 3; ++g) {
        double x = Z[(g + 1) * n + c];
        if (q->integrator == I_RUSH_LARSEN) {
          double e = exp(alpha[g] * dt);
          Z[(g + 1) * n + c] = x * e + (beta[g] / alpha[g]) * (e - 1.0);
        } else {
          Z[(g + 1) * n + c] = (x + dt * beta[g]) / (1.0 - dt * alpha[g]);
        }
      }
      Z[c] = u + dt * K1[c];
    }
  }
}

/* Advance `batch` independent states Z[batch][n_v][nz][ny][nx] by nsteps steps, in place (nz == 1:
 * the 2-D problem).  params == NULL: the default block.  Returns 0, or -1 on invalid arguments,
 * -2 on allocation failure. */
int oracle_step3d(int model, int nx, int ny, int nz, double dx, double dt, int scheme, int batch,
                  const double* params, double* Z, long long nsteps) {
  double pdef[32];
  problem q;
  q.model = model; q.stencil = scheme & 0xff; q.integrator = (scheme >> 8) & 0xff;
  q.boundary = (scheme >> 16) & 0xff; q.variant = (scheme >> 24) & 0xff;
  q.nx = nx; q.ny = ny; q.nz = nz; q.dx = dx; q.dt = dt;
  q.nv = oracle_num_fields(model);
  if (q.nv < 0) return -1;
  q.nd = num_diffusing(model);
  int r = (q.stencil == S_LAP9X4) ? 2 : 1;
  if (q.stencil > S_BOX9 || q.integrator > I_IMPLICIT_EULER || q.boundary > B_PERIODIC ||
      q.variant > V_TANHFREE) return -1;
  if (q.integrator >= I_RUSH_LARSEN && model != M_BOCF) return -1;
  if (nx < 2 * r + 1 || ny < 2 * r + 1 || batch < 1 || nsteps < 0) return -1;
  if (nz != 1 && (nz < 2 * r + 1 || q.stencil == S_BOX9)) return -1;
  if (!(dx > 0.0) || !(dt > 0.0) || !isfinite(dx) || !isfinite(dt)) return -1;
  if (params) q.p = params; else { oracle_default_params(model, pdef); q.p = pdef; }

  size_t n = (size_t)nx * ny * nz, N = n * q.nv;
  double* w = (double*)malloc(sizeof(double) * (5 * N + n));
  if (!w) return -2;
  for (int b = 0; b < batch; ++b)
    for (long long s = 0; s < nsteps; ++s) step_once(&q, Z + (size_t)b * N, w);
  free(w);
  return 0;
}

int oracle_step(int model, int nx, int ny, double dx, double dt, int scheme, int batch,
                const double* params, double* Z, long long nsteps) {
  return oracle_step3d(model, nx, ny, 1, dx, dt, scheme, batch, params, Z, nsteps);
}

/* Finite-difference Jacobian-vector products of the flow map:
 * J_b = (Z_b - Z_0)/eps for b = 1..batch-1, from already-integrated states Z[batch][N]. */
int oracle_jvp(const double* Z, int batch, size_t N, double eps, double* J) {
  if (batch < 2 || !(eps != 0.0)) return -1;
  for (int b = 1; b < batch; ++b)
    OMP_FOR
    for (long c = 0; c < (long)N; ++c) J[(size_t)(b - 1) * N + c] = (Z[(size_t)b * N + c] - Z[c]) / eps;
  return 0;
}
