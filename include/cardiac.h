/*
 * cardiac.h — C ABI of libcardiac.so: the fully explicit FP64 time step of the 2-D
 * reaction-diffusion system  dz/dt = D lap(z) + N[z]  (Eq. 1) with no-flux
 * boundaries (Eq. 2) for the FitzHugh-Nagumo (Eq. 3),
 * Karma (Eq. 4) and Bueno-Orovio-Cherry-Fenton (Eq. 5)
 * models, on one NVIDIA B200 (sm_100a).
 *
 * Everything behind this boundary is CUDA; there is no CPU fallback.  Every function that
 * touches the device fails with CARDIAC_ERR_CUDA when no usable device is present.
 *
 * Conventions
 *   - "state" is a dense float64 array [batch][n_v][ny][nx], x fastest (row-adjacent
 *     cells adjacent in memory).  Field order: FHN (u,v); Karma (u,v); BOCF (u,v,w,s).
 *   - Pointers are tagged host/device by an explicit int flag; device pointers must be valid
 *     on the CUDA device that was current when the context was created.
 *   - The caller owns every buffer it passes in (state arrays, the stream, a bound workspace)
 *     and must keep the stream and workspace alive until cardiac_destroy.  The library owns the
 *     context and anything it allocated itself.
 *   - cardiac_step and device-side set/get are enqueued on the context stream and return
 *     without synchronising; host-side set/get synchronise that stream before returning.
 *   - All functions returning int return CARDIAC_OK (0) or a negative error code;
 *     cardiac_last_error gives the text.  The library never checks stability (dt against
 *     dx^2/4D) nor NaN/Inf in the state.
 *   - step(a); step(b) is bitwise identical to step(a+b) as long as the same execution plan is
 *     used (cardiac_set_plan), results do not depend on the batch position of a member, and
 *     repeated runs are bitwise identical (no atomics on data, fixed summation order).
 */
#ifndef CARDIAC_H
#define CARDIAC_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct cardiac_ctx cardiac_ctx; /* opaque, owned by the library */

/* model ("three different models") */
enum { CARDIAC_FHN = 0, CARDIAC_KARMA = 1, CARDIAC_BOCF = 2 };

/* scheme = stencil | integrator | boundary | variant */
enum {
  /* bits 0-7: Laplacian stencil (Eq. 6).  dx = dy.      */
  CARDIAC_LAP5   = 0, /* Eq. 6 with alpha_a = 1, alpha_d = 0: (sum of 4 axial nbrs - 4 U)/dx^2 */
  CARDIAC_LAP9X4 = 1, /* radius-2 cross, per axis (-1,16,-30,16,-1)/(12 dx^2): the "larger stencil"
                         of PAPER.md:114, 4th order                                            */
  CARDIAC_BOX9   = 2, /* Eq. 6 with alpha_a = 2/3, alpha_d = 1/6, centre -10/3 (isotropic 3x3) */
  /* bits 8-15: time integrator.  Fixed dt.                                  */
  CARDIAC_EULER  = 0 << 8, /* z+ = z + dt f(z)                                                  */
  CARDIAC_HEUN   = 1 << 8, /* Y2 = z + dt f(z); z+ = z + dt/2 (f(z) + f(Y2))                    */
  CARDIAC_RK4    = 2 << 8, /* classic Runge-Kutta                                               */
  CARDIAC_RUSH_LARSEN   = 3 << 8, /* BOCF only: u by explicit Euler, gates x' = a x + b by the
                                     exponential update                      */
  CARDIAC_IMPLICIT_EULER = 4 << 8, /* BOCF only: u explicit, gates by pointwise implicit Euler  */
  /* bits 16-23: boundary condition                                                             */
  CARDIAC_NOFLUX   = 0 << 16, /* mirror about the boundary node: U[-m] = U[m], U[N-1+m] = U[N-1-m],
                                 each axis independently (PAPER.md:104 Fig. 1, :114)            */
  CARDIAC_PERIODIC = 1 << 16, /* "mapping to the opposite-edge values"           */
  /* bits 24-31: model variant                                                                  */
  CARDIAC_VARIANT_PAPER    = 0 << 24, /* equations as printed                                   */
  CARDIAC_VARIANT_TANHFREE = 1 << 24  /* tanh(x) -> 2 H_k'(x) - 1 (k' = param)     */
};

/* execution plan (how the same numbers are produced) */
enum {
  CARDIAC_PLAN_AUTO       = 0, /* library picks by (model, scheme, nx*ny*batch)                 */
  CARDIAC_PLAN_STAGE      = 1, /* one fused stencil+reaction+RK-stage launch per substep        */
  CARDIAC_PLAN_FUSED      = 2, /* all substeps of one time step (or several Euler steps) on chip,
                                  overlapped tiles, one launch                                  */
  CARDIAC_PLAN_PERSISTENT = 3, /* ONE launch for all nsteps: each batch member resident in the shared
                                  memory of a thread-block cluster (<= 16 CTAs), ghost rows pushed
                                  through distributed shared memory; grids up to C x 4096 cells
                                  (4-field model: C x 2048), C = 16 CTAs for batches of up to 4
                                  members, else 8; Euler, Heun, RK4                             */
  CARDIAC_PLAN_PAIR       = 4  /* two consecutive substeps per launch: the first on tile + ring into
                                  shared memory, the second from there (RK4: two launches, the fourth
                                  stage value never reaches memory; Heun: one launch; Euler: two time
                                  steps per launch); 2-D; Euler, Heun, RK4                      */
};

/* error codes */
enum {
  CARDIAC_OK = 0,
  CARDIAC_ERR_INVALID   = -1, /* invalid argument                                               */
  CARDIAC_ERR_CUDA      = -2, /* CUDA runtime error (text in cardiac_last_error)                */
  CARDIAC_ERR_NOSTATE   = -3, /* step/get_state before set_state                                */
  CARDIAC_ERR_WORKSPACE = -4  /* bound workspace too small or misaligned                        */
};

/* Number of fields n_v of a model: 2, 2, 4; -1 for an unknown model. */
int cardiac_num_fields(int model);

/* Number of entries of the model's parameter block (5, 9, 30); -1 for an unknown model.
 *   FHN  : D_u, delta(=D_v), epsilon, a1, a0
 *   Karma: gamma, tau_u, tau_v, u_h, u_v, u_star, Re, M, k
 *   BOCF : D, k, u_o, u_u, theta_v, theta_w, theta_v_minus, theta_o, tau_v1_minus, tau_v2_minus,
 *          tau_v_plus, tau_w1_minus, tau_w2_minus, k_w_minus, u_w_minus, tau_w_plus, tau_fi,
 *          tau_o1, tau_o2, tau_so1, tau_so2, k_so, u_so, tau_s1, tau_s2, k_s, u_s, tau_si,
 *          tau_w_inf, w_inf_star                                    (Q9) */
int cardiac_num_params(int model);

/* Copy the library's default parameter block of `model` into p[0..n-1] (host). n must equal
 * cardiac_num_params(model). */
int cardiac_default_params(int model, double* p, int n);

/* Create a context for `batch` independent states of nx*ny cells (N x N grid, spacing
 * dx = dy, fixed dt; nx != ny allowed).  Requires nx, ny >= 2r+1 (r = stencil radius), batch >= 1,
 * finite dx > 0 and dt > 0, known model/scheme bits, Rush-Larsen / implicit Euler only with BOCF.
 * The current CUDA device is captured.  Returns NULL on failure (text: cardiac_last_error(NULL)). */
cardiac_ctx* cardiac_create(int model, int nx, int ny, double dx, double dt, int scheme, int batch);

/* 3-D variant ("three-dimensional simulations (corresponding to ventricular tissue)";
 * DESIGN.md f4): nz planes of ny x nx cells, spacing dx in all three directions; the stencil bits
 * select the same per-axis weights applied along x, y and z (CARDIAC_LAP5 -> 7-point, CARDIAC_LAP9X4
 * -> 13-point 4th-order cross; CARDIAC_BOX9 is 2-D only), the boundary rule applies per axis.  State
 * layout: dense [batch][n_v][nz][ny][nx].  nz == 1 is cardiac_create(); otherwise nz >= 2r+1 and
 * batch * nz <= 65535.  3-D contexts run plan STAGE. */
cardiac_ctx* cardiac_create3d(int model, int nx, int ny, int nz, double dx, double dt, int scheme, int batch);

/* Replace the model parameters (host array, n == cardiac_num_params(model)).  Takes effect for
 * subsequent steps.  M (Karma) must be an integer in [1, 16]. */
int cardiac_set_params(cardiac_ctx*, const double* p, int n);

/* Read back the active parameter block (host array). */
int cardiac_get_params(const cardiac_ctx*, double* p, int n);

/* Use `cuda_stream` (a cudaStream_t passed as void*, e.g. torch.cuda.current_stream().cuda_stream;
 * NULL = legacy default stream) for all subsequent work. */
int cardiac_set_stream(cardiac_ctx*, void* cuda_stream);

/* Choose the execution plan (CARDIAC_PLAN_*).  CARDIAC_ERR_INVALID if the plan does not support the context's
 * (model, scheme, size).  Every plan and implementation gives the same numbers (bitwise between implementations of
 * a plan; to roundoff between plans).  `param` is plan specific:
 *   STAGE      0 = by size, 1 = DIRECT (every thread loads its own operands), 2 = RING (persistent CTAs fed by a TMA
 *              shared-memory ring)
 *   PAIR       0 = by size, 1 = DIRECT, 2 = TMA (persistent CTAs, operands by box copies one tile ahead)
 *   FUSED      Euler: time steps per launch (0 = default 4, or 1);  Heun / RK4: window + 16 x implementation with
 *              window 0 = by size, 1 = 80x48 cells (one CTA per SM), 2 = 48x40 (two CTAs per SM; two-field models),
 *              3 / 4 / 5 = 64x56 / 64x48 / 56x48, 7 = 64x56 on 896 threads and 8 = 64x32 on 1024 threads (two-field
 *              models, RK4), and
 *              implementation 0 = by size, 1 = one CTA per tile, 2 = TMA (persistent CTAs whose windows arrive one
 *              tile ahead; two-field models, windows 1, 2, 3, 7, grids larger than window + halo)
 *   PERSISTENT 0
 * AUTO: PERSISTENT below ~128x128 .. 192x192 cells per member (by model and integrator; batches of up to 4 members,
 * half of that up to 16); FUSED for the two-field models (TMA implementation from ~370 - 450 tiles) and for a 4-field
 * grid that is one wave of its tiles; PAIR (TMA) for the 4-field model with RK4 from 1024^2 cells (Heun: 1536^2) and
 * below that where its 64 x 24 tiles fill whole rounds of the persistent grid; STAGE for Karma + Euler below 2048^2
 * (except one-wave grids) and everything else.  DESIGN.md "Plan choice" has the measurements. */
int cardiac_set_plan(cardiac_ctx*, int plan, int param);

/* The plan that cardiac_step will use (resolved from AUTO). */
int cardiac_get_plan(const cardiac_ctx*);

/* Bytes of device workspace the context needs (all stage buffers and halos). */
size_t cardiac_workspace_bytes(const cardiac_ctx*);

/* Bind caller-allocated device memory (256-byte aligned, >= cardiac_workspace_bytes) as the
 * workspace; must be called before the first set_state, else the library cudaMallocs its own. */
int cardiac_bind_workspace(cardiac_ctx*, void* dev_ptr, size_t bytes);

/* Copy a dense [batch][n_v][ny][nx] float64 state into the context. src_on_device != 0: src is a
 * device pointer, the copy is enqueued on the stream.  Otherwise src is a host pointer and the call
 * returns after the copy completed. */
int cardiac_set_state(cardiac_ctx*, const double* src, int src_on_device);

/* Advance every batch member by nsteps time steps of size dt.  nsteps == 0 is a no-op, nsteps < 0
 * is invalid.  Asynchronous on the context stream. */
int cardiac_step(cardiac_ctx*, long long nsteps);

/* Copy the current state out, layout as in set_state. */
int cardiac_get_state(cardiac_ctx*, double* dst, int dst_on_device);

/* Finite-difference Jacobian-vector products of the flow map: with member 0 the
 * base trajectory phi(x) and members b = 1..batch-1 the perturbed ones phi(x + eps v_b), write
 * J_b = (phi(x + eps v_b) - phi(x)) / eps as dense [batch-1][n_v][ny][nx] float64 into dst. */
int cardiac_get_jvp(cardiac_ctx*, double eps, double* dst, int dst_on_device);

/* Row-slab decomposition of ONE grid across GPUs (the paper is single-GPU,
 * PAPER.md:122).  A rank holds a context over its rows PLUS g ghost rows towards each neighbour, with
 * g = radius x substeps per time step x time steps between exchanges: information travels one stencil
 * radius per substep, so after those time steps the rank's own rows are exactly the
 * single-grid result and only the ghost rows are stale.  The exchange reads the g own rows next to the
 * cut and writes them into the neighbour's ghost rows with these two calls:
 *   cardiac_get_rows  rows [j0, j0+nrows) of every field of every batch member -> dense
 *                     [batch][n_v][nrows][nx] float64 at dst.  A DEVICE dst may be any address the
 *                     GPU can store to, including peer memory mapped over NVLink (the pack kernel
 *                     then is the transfer); asynchronous on the context stream.
 *   cardiac_set_rows  the reverse.
 * For 3-D contexts a "row" is an index of the flattened (plane, row) pair, so a slab of planes is a
 * row range too.  Host buffers synchronise the stream.  CARDIAC_ERR_INVALID when the range leaves
 * the grid, CARDIAC_ERR_NOSTATE before set_state. */
int cardiac_get_rows(cardiac_ctx*, int j0, int nrows, double* dst, int dst_on_device);
int cardiac_set_rows(cardiac_ctx*, int j0, int nrows, const double* src, int src_on_device);

/* Text of the last error on this context; ctx == NULL: the calling thread's last create() error.
 * Never NULL; empty string when there was none. */
const char* cardiac_last_error(const cardiac_ctx*);

void cardiac_destroy(cardiac_ctx*);

#ifdef __cplusplus
}
#endif
#endif /* CARDIAC_H */
