// api.cu — the C ABI of include/cardiac.h: context, validation, workspace, plan selection,
// CUDA-graph capture of the per-step launch sequence, state copies.  No arithmetic of the method
// lives here; it only sequences the kernels of *_kernels.cu.
#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>
#include <string>

#include "../../include/cardiac.h"
#include "../../include/cardiac_diag.h"
#include "plans.h"
#include "stage.cuh"

using namespace cardiac;

namespace {
thread_local std::string g_create_error;

constexpr int kMaxBuf = 4;
constexpr int kGraphNodes = 64;  // kernel nodes per captured graph
}  // namespace

struct cardiac_ctx {
  Problem pb{};
  int scheme = 0;
  int nparams = 0;
  int device = 0;
  cudaStream_t stream = nullptr;
  cudaStream_t cap_stream = nullptr;  // only ever used in capture mode
  int plan_req = CARDIAC_PLAN_AUTO, plan = CARDIAC_PLAN_STAGE, plan_param = 0;
  int fused_impl = 0;   // plan FUSED: 0 = by size, 1 = one CTA per tile, 2 = persistent CTAs fed by TMA
  void* ws = nullptr;
  size_t ws_bytes = 0;
  bool ws_owned = false;
  int nbuf = 0;
  double* buf[kMaxBuf] = {nullptr, nullptr, nullptr, nullptr};
  int cur = 0;  // buffer holding the state
  bool has_state = false;
  cudaGraphExec_t graph[kMaxBuf] = {nullptr, nullptr, nullptr, nullptr};  // keyed by `cur` at graph start
  int graph_steps = 0;
  long long launches = 0;
  std::string err;
};

namespace {

int fail(cardiac_ctx* c, int code, const std::string& msg) {
  if (c) c->err = msg;
  return code;
}
int fail_cuda(cardiac_ctx* c, cudaError_t e, const char* what) {
  return fail(c, CARDIAC_ERR_CUDA, std::string(what) + ": " + cudaGetErrorString(e));
}
#define CK(call)                                                  \
  do {                                                            \
    cudaError_t e_ = (call);                                      \
    if (e_ != cudaSuccess) return fail_cuda(c, e_, #call);        \
  } while (0)

int stages_of(int integ) { return integ == I_HEUN ? 2 : (integ == I_RK4 ? 4 : 1); }
int buffers_of(int integ) { return integ == I_RK4 ? 4 : 2; }

size_t buffer_doubles(const Problem& pb) { return (size_t)pb.bstride * pb.batch; }

void drop_graphs(cardiac_ctx* c) {
  for (auto& g : c->graph)
    if (g) { cudaGraphExecDestroy(g); g = nullptr; }
  c->graph_steps = 0;
}

void carve(cardiac_ctx* c) {
  size_t n = buffer_doubles(c->pb);
  for (int b = 0; b < c->nbuf; ++b) c->buf[b] = (double*)c->ws + b * n;
}

// AUTO: the on-chip tile engine wherever a time step is cheap enough per cell that the global
// round trip per substep dominates (FHN, Karma); the 4-field ionic model is FP64-pipe bound and its
// register-resident patches are too small to amortise an 8-cell halo, so it stays stage-synchronous
// (DESIGN.md "Plans").
// FUSED + Heun/RK4: which window.  1 = 80 x 48 cells, 3 = 64 x 56, 4 = 64 x 48, 5 = 56 x 48 (one CTA per SM;
// 3-5: RK4 of the two-field models), 2 = 48 x 40 (two CTAs per SM; two-field models).  Measured on B200
// (Karma LAP5 RK4 and FHN LAP9X4 RK4, 362^2 - 1536^2, every window forced):
//  * one CTA per SM: the CTAs of a wave run in lock step and a time step costs (waves) x (CTA lifetime),
//    the lifetime being a fixed part (launch, window load, barriers, store) worth ~2000 cells plus the
//    window area — 10.3 / 10.0 / 8.8 / 8.6 us per wave for windows 1 / 3 / 4 / 5 (Karma), 7.0 / 6.5 / 5.6 /
//    5.4 us (FHN).  The window whose tiles fill whole waves wins: 512^2 with a halo of 8 is one wave of
//    143 CTAs of window 3 (7.0 us) or of 128 of window 1 (7.4 us), but two waves of window 4 (11.1 us).
//  * two small CTAs per SM run out of step: time grows linearly with their number n, 0.57 + n/296
//    waves of 1/1.18 of window 1's wave time.  With a halo of 8 the small window has 40 % useful cells
//    against 53 % and only wins when the whole grid is one CTA per SM (<= 256^2: 7.7 -> 6.3 us per step).
int fused_window_auto(const Problem& pb) {
  if (pb.nv > 2 || pb.integrator == I_EULER) return 1;
  const int H = pb.radius * stages_of(pb.integrator);
  // Karma, RK4, halo 4: the 64 x 56 window on 896 threads, TMA-fed, from ~400 tiles (1024^2); measured above
  if (pb.model == CARDIAC_KARMA && pb.integrator == I_RK4 && H <= 4 && fused_tma_supported(pb, 7, 1)) {
    const long long n7 = (long long)((pb.nx + 55) / 56) * ((pb.ny + 47) / 48) * pb.batch;
    if (n7 >= 400) return 7;
  }
  auto ctas = [&](long long ew, long long eh) {
    const long long tw = ew - 2 * H, th = eh - 2 * H;
    return ((pb.nx + tw - 1) / tw) * ((pb.ny + th - 1) / th) * pb.batch;
  };
  // one wave of 64 x 32 windows on 1024 threads (one row of a pair per thread): the shortest CTA lifetime for a
  // halo of 8 and for Karma (tile_dispatch.cuh, window 8)
  if (pb.integrator == I_RK4 && (H == 8 || pb.model == CARDIAC_KARMA) && 64 - 2 * H > 0 && 32 - 2 * H > 0 &&
      ctas(64, 32) <= 148)
    return 8;
  const long long small = ctas(48, 40);
  if (small <= 148) return 2;
  constexpr double kFixed = 2000.0;   // cells
  auto cost = [&](long long ew, long long eh) {
    return (double)((ctas(ew, eh) + 147) / 148) * ((double)(ew * eh) + kFixed);
  };
  int best = 1;
  double best_cost = cost(80, 48);
  if (pb.integrator == I_RK4) {
    const double c3 = cost(64, 56), c4 = cost(64, 48), c5 = cost(56, 48);
    if (c3 < best_cost) { best = 3; best_cost = c3; }
    if (c4 < best_cost) { best = 4; best_cost = c4; }
    if (c5 < best_cost) { best = 5; best_cost = c5; }
  }
  // (not for FHN + Heun, two diffusing fields at halo 4: measured, the 80 x 48 window wins at every size above one wave
  // of small windows — 448^2 5.6 against 6.4 us per step, 768^2 9.5 / 11.0)
  if (H <= 4 && !(pb.model == CARDIAC_FHN && pb.integrator == I_HEUN)) {
    const double c2 = (80.0 * 48.0 + kFixed) / 1.18 * (0.57 + (double)small / 296.0);
    if (c2 < best_cost) best = 2;
  }
  return best;
}

int auto_plan(const Problem& pb) {
  const bool rk_like = pb.integrator == I_EULER || pb.integrator == I_HEUN || pb.integrator == I_RK4;
  // a grid that fits one SM never leaves it: the paper's launch-bound regime N < N0
  if (pb.nz > 1) return CARDIAC_PLAN_STAGE;   // 3-D: the stage-synchronous plan only
  if (resident_preferred(pb)) return CARDIAC_PLAN_PERSISTENT;
  const long long pair_tiles = (long long)((pb.nx + 63) / 64) * ((pb.ny + 23) / 24) * pb.batch;
  // (Heun of the two-field models: plan PAIR / TMA was ahead of FUSED for FHN LAP9X4 until the FUSED / TMA pipeline lost
  // its end-of-tile barrier; since then the 80 x 48 window fed by TMA wins from 1024^2 — 2048^2 46.3 against 51.0 us per
  // step, 4096^2 148 / 186 = 113 / 90 Gcell-step/s — and FUSED is taken below)
  // Karma + forward Euler: the exponential makes a substep too expensive to recompute over the halo of four
  // blocked steps; one launch per step wins up to 1536^2 (round 2, LAP5, STAGE / FUSED x 4: 256^2 32 / 26, 1024^2
  // 187 / 147, 1536^2 220 / 188 Gcell-step/s; from 2048^2 the TMA-fed FUSED is ahead, 180 / 171, 4096^2 205 / 183)
  // ... except where the grid is ONE wave of 80 x 48 windows with at least 60 tiles (362^2 .. 640^2: 640^2 2.7 against
  // 4.3 us per step, 448^2 2.64 / 2.78; below, the two are within 3 %)
  if (pb.model == CARDIAC_KARMA && pb.integrator == I_EULER && (long long)pb.nx * pb.ny * pb.batch < (1LL << 22)) {
    const int H = pb.radius * kEulerBlock, tw = 80 - 2 * H, th = 48 - 2 * H;
    const long long tiles = tw > 0 && th > 0 ? (long long)((pb.nx + tw - 1) / tw) * ((pb.ny + th - 1) / th) * pb.batch : 0;
    return tiles >= 60 && tiles <= 148 ? CARDIAC_PLAN_FUSED : CARDIAC_PLAN_STAGE;
  }
  // Karma with a radius-2 stencil: every cell of the halo pays an exponential, so beyond one wave of windows the
  // stage-synchronous plan wins while its buffers stay in L2 (round 2 audit, LAP9X4: RK4 1024^2 30.1 against 37.7 us
  // per step, Heun 1536^2 26.8 / 36.2, 768^2 9.6 / 11.6; from 1536^2 / 2048^2 the TMA-fed FUSED is ahead again), and
  // four blocked Euler steps (halo 8) never pay beyond one wave (4096^2 96 / 118)
  if (pb.model == CARDIAC_KARMA && pb.radius >= 2 && rk_like) {
    const int H = pb.radius * (pb.integrator == I_RK4 ? 4 : (pb.integrator == I_HEUN ? 2 : kEulerBlock));
    auto ctas = [&](int ew, int eh) -> long long {
      const int tw = ew - 2 * H, th = eh - 2 * H;
      if (tw <= 0 || th <= 0) return 1LL << 40;
      return (long long)((pb.nx + tw - 1) / tw) * ((pb.ny + th - 1) / th) * pb.batch;
    };
    const long long cells = (long long)pb.nx * pb.ny * pb.batch;
    long long one_wave = ctas(80, 48);
    if (pb.integrator != I_EULER) one_wave = std::min(one_wave, ctas(48, 40));
    if (pb.integrator == I_RK4) one_wave = std::min(std::min(one_wave, ctas(64, 56)), ctas(64, 32));
    bool fused = one_wave <= 148;
    // (Heun: one wave of the LARGE window costs ~6.8 us, more than two stage launches below ~575^2)
    if (pb.integrator == I_HEUN && ctas(48, 40) > 148 && cells < 330000) fused = false;
    if (fused) return CARDIAC_PLAN_FUSED;
    const long long working_set = cells * pb.nv * 8 * (pb.integrator == I_RK4 ? 4 : 2);
    if (pb.integrator == I_EULER || working_set <= (96LL << 20)) return CARDIAC_PLAN_STAGE;
    // streaming sizes: a pair's ring of r cells against the window's halo of 2r / 4r (2048^2 Heun 58.5 against 62.7 us per
    // step, 4096^2 RK4 479 / 511)
    if (pair_tiles >= 4 * kPairTMinTiles && pair_tma_supported(pb)) return CARDIAC_PLAN_PAIR;
    return CARDIAC_PLAN_FUSED;
  }
  if (rk_like && pb.model != CARDIAC_BOCF) return CARDIAC_PLAN_FUSED;
  // 4-field model: two substeps per launch once the grid gives every SM enough tiles (measured on B200,
  // RK4 1536^2 +2 %, 2048^2 +6 %, 4096^2 +15 %, 8192^2 +19 % over STAGE, behind at
  // 1024^2; Heun +2 % at 4096^2, behind at 2048^2)
  if (pb.model == CARDIAC_BOCF) {
    // a grid that is ONE wave of the 4-field model's fused tiles (48 x 32 window) costs one CTA lifetime per time
    // step instead of four launch-bound stage launches (round 2, LAP9X4 RK4: 256^2 9.6 against 14.4 us per step;
    // two waves already lose: 362^2 18.5 against 16.5)
    // (the same for Heun, halo 2 r, and for four blocked Euler steps, halo 4 r — LAP9X4: Euler 256^2 2.3 against 3.2 us
    // per step, 320^2 = two waves 4.2 / 3.5; Heun 320^2 6.6 / 7.1, 362^2 = two waves 11.6 / 7.8)
    if (rk_like) {
      const int H = pb.radius * (pb.integrator == I_HEUN ? 2 : 4), tw = 48 - 2 * H, th = 32 - 2 * H;
      if (tw > 0 && th > 0 && (long long)((pb.nx + tw - 1) / tw) * ((pb.ny + th - 1) / th) * pb.batch <= 148)
        return CARDIAC_PLAN_FUSED;
    }
    const long long cells = (long long)pb.nx * pb.ny * pb.batch;
    if ((pb.integrator == I_RK4 && cells >= kPairMinCellsRK4) || (pb.integrator == I_HEUN && cells >= kPairMinCellsHeun))
      return CARDIAC_PLAN_PAIR;
    // the TMA-fed implementation already wins once every persistent CTA has four tiles to pipeline
    // (round 2, LAP9X4 RK4: 1024^2 15.5 against 13.0 Gcell-step/s, 768^2 14.0 against 14.8)
    if (pb.integrator == I_RK4 && pair_tiles >= kPairTMinTiles && pair_tma_supported(pb)) return CARDIAC_PLAN_PAIR;
    // ... and below that where the tiles fill whole rounds of the persistent grid (plans.h; Heun: up to two rounds —
    // 448^2 7.8 against 9.7 us per step, 640^2 13.0 / 14.9, but 896^2 23.5 / 23.2)
    if ((pb.integrator == I_RK4 || pb.integrator == I_HEUN) && pair_tma_supported(pb) &&
        pair_tma_fills_rounds(pair_tiles, pb.integrator == I_RK4 ? 4 : 2))
      return CARDIAC_PLAN_PAIR;
    // Heun: 2048^2 40.4 against 36.8 (STAGE), 1536^2 63.2 against 69.8 us per step, 1024^2 36.6 against 38.0
    if (pb.integrator == I_HEUN && pair_tiles >= 2 * kPairTMinTiles && pair_tma_supported(pb)) return CARDIAC_PLAN_PAIR;
  }
  return CARDIAC_PLAN_STAGE;
}

// FUSED + Heun/RK4: plan_param = window (set_plan resolves 0)
int fused_window(const cardiac_ctx* c) {
  return (c->plan == CARDIAC_PLAN_FUSED && c->pb.integrator != I_EULER) ? c->plan_param : 1;
}

// Plan FUSED: one launch advances `ksteps` time steps (1, or kEulerBlock Euler steps), ping-pong.
int enqueue_fused(cardiac_ctx* c, cudaStream_t s, int ksteps) {
  const int other = c->cur == 0 ? 1 : 0;   // (plan PAIR may have left the state in buffer 2)
  TileLaunch tl{c->buf[c->cur], c->buf[other], ksteps, c->fused_impl, fused_window(c)};
  bool tma = false;
  if (c->fused_impl != 1 && fused_tma_supported(c->pb, tl.window, ksteps)) {
    if (c->fused_impl == 2) {
      tma = true;
    } else {   // AUTO: once every persistent CTA has several tiles to pipeline
      const int ns = c->pb.integrator == I_RK4 ? 4 : (c->pb.integrator == I_HEUN ? 2 : ksteps);
      int tw, th;
      fused_tile_of(c->pb.integrator == I_EULER ? 1 : tl.window, c->pb.radius * ns, tw, th);
      const long long ntiles = (long long)((c->pb.nx + tw - 1) / tw) * ((c->pb.ny + th - 1) / th) * c->pb.batch;
      tma = tl.window == 7 ? ntiles >= 400 : ntiles >= kFusedTMinTiles * (tl.window == 2 ? 2 : 1);
      // Heun, 80 x 48 window: two substeps per tile leave less to overlap, the pipeline pays from ~2.5 tiles per CTA
      // (FHN LAP9X4: 1024^2 = 390 tiles 13.3 against 14.2 us per step, 896^2 = 299 tiles 13.4 / 13.5, 768^2 9.9 / 9.5)
      if (c->pb.integrator == I_HEUN && tl.window == 1) tma = ntiles >= 370;
    }
  }
  cudaError_t e = tma ? launch_fusedt(c->pb, tl, s) : launch_fused(c->pb, tl, s);
  if (e != cudaSuccess) return fail_cuda(c, e, "fused launch");
  c->launches++;
  c->cur = other;
  return CARDIAC_OK;
}

// Plan PAIR: which implementation runs (bitwise identical results): DIRECT (pair.cuh) or TMA (pairt.cuh)
bool pair_uses_tma(const cardiac_ctx* c) {
  const Problem& pb = c->pb;
  if (pb.pair_impl == 1 || !pair_tma_supported(pb)) return false;
  if (pb.pair_impl == 2) return true;
  const long long ntiles = (long long)((pb.nx + 63) / 64) * ((pb.ny + 23) / 24) * pb.batch;
  if (pb.model == CARDIAC_BOCF && (pb.integrator == I_RK4 || pb.integrator == I_HEUN) &&
      pair_tma_fills_rounds(ntiles, pb.integrator == I_RK4 ? 4 : 2))
    return true;   // auto_plan's mid-size rule for the 4-field model
  return ntiles >= kPairTMinTiles;
}

// ... TMA implementation: one time step (Heun, RK4) or two (Euler)
int enqueue_pair_tma(cardiac_ctx* c, cudaStream_t s) {
  const Problem& pb = c->pb;
  const double dt = pb.dt;
  const int ring = pb.integrator == I_RK4 ? 3 : 2;
  const int n1 = c->cur < ring ? (c->cur + 1) % ring : 0, n2 = (n1 + 1) % ring;
  double* b0 = c->buf[c->cur];
  double* b1 = c->buf[n1];
  auto go = [&](const PairTLaunch& pl) -> int {
    cudaError_t e = launch_pairt(pb, pl, s);
    if (e != cudaSuccess) return fail_cuda(c, e, "pair (TMA) launch");
    c->launches++;
    return CARDIAC_OK;
  };
  int rc = CARDIAC_OK;
  PairTLaunch pl{};
  pl.in = b0; pl.y = b0;
  switch (pb.integrator) {
    case I_EULER:
      pl.ka = K_SELF; pl.kb = K_SELF; pl.out = b1; pl.a_wf = dt; pl.w_f = dt;
      rc = go(pl);
      break;
    case I_HEUN:
      pl.ka = K_SELF; pl.kb = K_BASE; pl.out = b1; pl.a_wf = dt;
      pl.w_y = 0.5; pl.w_in = 0.5; pl.w_f = 0.5 * dt;
      rc = go(pl);
      break;
    case I_RK4: {   // the combinations and weights of plan STAGE (enqueue_step); P takes Y2's place in memory
      double* b2 = c->buf[n2];
      pl.ka = K_SELF; pl.kb = K_BASE; pl.out = b2; pl.out2 = b1; pl.a_wf = 0.5 * dt;
      pl.w_y = 1.0; pl.w_in = 0.0; pl.w_f = 0.5 * dt;
      pl.p_wy = -1.0 / 3.0; pl.p_wA = 1.0 / 3.0; pl.p_wB = 2.0 / 3.0;
      if ((rc = go(pl))) break;
      pl = PairTLaunch{};
      pl.ka = K_BASE; pl.kb = K_RK4F; pl.in = b2; pl.y = b0; pl.P = b1; pl.out = b1;
      pl.a_wy = 1.0; pl.a_win = 0.0; pl.a_wf = dt;
      pl.w_in = 1.0 / 3.0; pl.w_f = dt / 6.0;
      rc = go(pl);
      break;
    }
    default:
      return fail(c, CARDIAC_ERR_INVALID, "PAIR supports Euler, Heun and RK4 only");
  }
  if (rc) return rc;
  c->cur = n1;
  return CARDIAC_OK;
}

// Plan PAIR: buffers the state rotates through (RK4: y, Y2, Y3 — Y4 never leaves the SM)
int pair_ring(const cardiac_ctx* c) { return c->pb.integrator == I_RK4 ? 3 : 2; }

// Plan PAIR: one time step (Heun, RK4) or two (Euler) in one or two launches of two substeps each.
int enqueue_pair(cardiac_ctx* c, cudaStream_t s) {
  if (pair_uses_tma(c)) return enqueue_pair_tma(c, s);
  const Problem& pb = c->pb;
  const double dt = pb.dt;
  const int ring = pair_ring(c);
  const int n1 = c->cur < ring ? (c->cur + 1) % ring : 0, n2 = (n1 + 1) % ring;
  double* b0 = c->buf[c->cur];
  double* b1 = c->buf[n1];
  auto go = [&](const PairLaunch& pl) -> int {
    cudaError_t e = launch_pair(pb, pl, s);
    if (e != cudaSuccess) return fail_cuda(c, e, "pair launch");
    c->launches++;
    return CARDIAC_OK;
  };
  int rc = CARDIAC_OK;
  PairLaunch pl{};
  pl.in = b0; pl.y = b0;
  switch (pb.integrator) {
    case I_EULER:   // y1 = y + dt f(y) [on chip]; y2 = y1 + dt f(y1)
      pl.ka = K_SELF; pl.kb = K_SELF; pl.out = b1; pl.a_wf = dt; pl.w_f = dt;
      rc = go(pl);
      break;
    case I_HEUN:    // Y2 = y + dt f(y) [on chip]; y+ = (y + Y2)/2 + dt/2 f(Y2)
      pl.ka = K_SELF; pl.kb = K_BASE; pl.out = b1; pl.a_wf = dt;
      pl.w_y = 0.5; pl.w_in = 0.5; pl.w_f = 0.5 * dt;
      rc = go(pl);
      break;
    case I_RK4: {   // same combinations and weights as plan STAGE (enqueue_step)
      double* b2 = c->buf[n2];
      pl.ka = K_SELF; pl.kb = K_BASE; pl.mid = b1; pl.out = b2; pl.a_wf = 0.5 * dt;
      pl.w_y = 1.0; pl.w_in = 0.0; pl.w_f = 0.5 * dt;
      if ((rc = go(pl))) break;
      pl = PairLaunch{};
      pl.ka = K_BASE; pl.kb = K_RK4F; pl.in = b2; pl.y = b0; pl.A = b1; pl.B = b2; pl.out = b1;
      pl.a_wy = 1.0; pl.a_win = 0.0; pl.a_wf = dt;
      pl.w_y = -1.0 / 3.0; pl.w_in = 1.0 / 3.0; pl.w_A = 1.0 / 3.0; pl.w_B = 2.0 / 3.0; pl.w_f = dt / 6.0;
      rc = go(pl);
      break;
    }
    default:
      return fail(c, CARDIAC_ERR_INVALID, "PAIR supports Euler, Heun and RK4 only");
  }
  if (rc) return rc;
  c->cur = n1;
  return CARDIAC_OK;
}

// time steps advanced by one repetition unit of the plan
int unit_steps(const cardiac_ctx* c) {
  if (c->plan == CARDIAC_PLAN_PAIR) return c->pb.integrator == I_EULER ? 2 : 1;
  return (c->plan == CARDIAC_PLAN_FUSED && c->pb.integrator == I_EULER) ? c->plan_param : 1;
}

// one repetition unit of the plan (unit_steps time steps)
int enqueue_step(cardiac_ctx* c, cudaStream_t s);
int enqueue_unit(cardiac_ctx* c, cudaStream_t s) {
  if (c->plan == CARDIAC_PLAN_PAIR) return enqueue_pair(c, s);
  const int us = unit_steps(c);
  return us == 1 ? enqueue_step(c, s) : enqueue_fused(c, s, us);
}

// Enqueue the kernels of ONE time step on `s`; advances c->cur as the real execution would.
int enqueue_step(cardiac_ctx* c, cudaStream_t s) {
  if (c->plan == CARDIAC_PLAN_FUSED) return enqueue_fused(c, s, 1);
  if (c->plan == CARDIAC_PLAN_PAIR && c->pb.integrator != I_EULER) return enqueue_pair(c, s);
  const Problem& pb = c->pb;
  const double dt = pb.dt;
  StageLaunch st{};
  auto go = [&](int kind, const double* in, const double* y, const double* A, const double* B,
                double* out, double w_y, double w_in, double w_A, double w_B, double w_f) -> int {
    st.kind = kind; st.in = in; st.y = y; st.A = A; st.B = B; st.out = out;
    st.w_y = w_y; st.w_in = w_in; st.w_A = w_A; st.w_B = w_B; st.w_f = w_f;
    cudaError_t e = launch_stage(pb, st, s);
    if (e != cudaSuccess) return fail_cuda(c, e, "stage launch");
    c->launches++;
    return CARDIAC_OK;
  };
  int rc = CARDIAC_OK;
  // b[0] holds the state; b[1..] are the other buffers (the state may sit in buffer 1 after an
  // odd number of ping-pong launches)
  double* b[kMaxBuf];
  b[0] = c->buf[c->cur];
  for (int i = 0, n = 1; i < c->nbuf; ++i)
    if (i != c->cur) b[n++] = c->buf[i];
  switch (pb.integrator) {
    case I_EULER:
    case I_RUSH_LARSEN:
    case I_IMPLICIT_EULER: {
      int kind = pb.integrator == I_EULER ? K_SELF : (pb.integrator == I_RUSH_LARSEN ? K_RL : K_IE);
      rc = go(kind, b[0], nullptr, nullptr, nullptr, b[1], 0, 0, 0, 0, dt);
      for (int i = 0; i < c->nbuf; ++i)
        if (c->buf[i] == b[1]) c->cur = i;
      break;
    }
    case I_HEUN:
      // Y2 = y + dt f(y);  y+ = (y + Y2)/2 + dt/2 f(Y2)   [= y + dt/2 (f(y) + f(Y2))]
      if ((rc = go(K_SELF, b[0], nullptr, nullptr, nullptr, b[1], 0, 0, 0, 0, dt))) break;
      rc = go(K_BASE, b[1], b[0], nullptr, nullptr, b[0], 0.5, 0.5, 0, 0, 0.5 * dt);
      break;
    case I_RK4:
      // Y2 = y + dt/2 f(y); Y3 = y + dt/2 f(Y2); Y4 = y + dt f(Y3);
      // y+ = (Y2 + 2 Y3 + Y4 - y)/3 + dt/6 f(Y4)   [accumulator-free classic RK4]
      if ((rc = go(K_SELF, b[0], nullptr, nullptr, nullptr, b[1], 0, 0, 0, 0, 0.5 * dt))) break;
      if ((rc = go(K_BASE, b[1], b[0], nullptr, nullptr, b[2], 1.0, 0.0, 0, 0, 0.5 * dt))) break;
      if ((rc = go(K_BASE, b[2], b[0], nullptr, nullptr, b[3], 1.0, 0.0, 0, 0, dt))) break;
      rc = go(K_RK4F, b[3], b[0], b[1], b[2], b[0], -1.0 / 3.0, 1.0 / 3.0, 1.0 / 3.0, 2.0 / 3.0,
              dt / 6.0);
      break;
    default:
      rc = fail(c, CARDIAC_ERR_INVALID, "unknown integrator");
  }
  return rc;
}

// Capture `units` repetition units starting from parity `cur` into an executable graph.
int build_graph(cardiac_ctx* c, int units) {
  int parity = c->cur;
  long long launches_before = c->launches;
  CK(cudaStreamBeginCapture(c->cap_stream, cudaStreamCaptureModeThreadLocal));
  int rc = CARDIAC_OK;
  for (int s = 0; s < units && rc == CARDIAC_OK; ++s) rc = enqueue_unit(c, c->cap_stream);
  const int end_cur = c->cur;
  cudaGraph_t g = nullptr;
  cudaError_t e = cudaStreamEndCapture(c->cap_stream, &g);
  c->cur = parity;  // capture executed nothing
  c->launches = launches_before;
  if (rc != CARDIAC_OK) { if (g) cudaGraphDestroy(g); return rc; }
  if (e != cudaSuccess) return fail_cuda(c, e, "cudaStreamEndCapture");
  if (end_cur != parity) {   // a graph is replayed back to back: it must end in the buffer it started from
    cudaGraphDestroy(g);
    return fail(c, CARDIAC_ERR_INVALID, "internal: graph does not return to its start buffer");
  }
  e = cudaGraphInstantiate(&c->graph[parity], g, 0);
  cudaGraphDestroy(g);
  if (e != cudaSuccess) return fail_cuda(c, e, "cudaGraphInstantiate");
  c->graph_steps = units;
  return CARDIAC_OK;
}

int ensure_workspace(cardiac_ctx* c) {
  if (c->ws) return CARDIAC_OK;
  size_t bytes = cardiac_workspace_bytes(c);
  CK(cudaMalloc(&c->ws, bytes));
  c->ws_bytes = bytes;
  c->ws_owned = true;
  carve(c);
  return CARDIAC_OK;
}

// Between two cardiac_step calls only buf[cur] holds data; every other stage buffer is free.  Host-side
// get_jvp / get_rows / set_rows stage their dense payload there (never larger than a pitched state
// buffer), so the exchange path allocates nothing and implies no device-wide synchronisation.
double* scratch_buffer(const cardiac_ctx* c) { return c->buf[(c->cur + 1) % c->nbuf]; }

struct DeviceGuard {
  int prev = -1;
  explicit DeviceGuard(int dev) {
    if (cudaGetDevice(&prev) != cudaSuccess) prev = -1;
    if (prev != dev) cudaSetDevice(dev);
    else prev = -1;
  }
  ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};

}  // namespace

extern "C" {

int cardiac_num_fields(int model) {
  switch (model) {
    case CARDIAC_FHN: return 2;
    case CARDIAC_KARMA: return 2;
    case CARDIAC_BOCF: return 4;
  }
  return -1;
}

int cardiac_num_params(int model) {
  switch (model) {
    case CARDIAC_FHN: return 5;
    case CARDIAC_KARMA: return 9;
    case CARDIAC_BOCF: return 30;
  }
  return -1;
}

int cardiac_default_params(int model, double* p, int n) {
  if (!p || n != cardiac_num_params(model)) return CARDIAC_ERR_INVALID;
  // FHN: PAPER.md:54.  Karma: PAPER.md:63 + Ref. [2] values (Q7).  BOCF: PAPER.md:76,
  // epicardial set of Ref. [3] (Q9), D in cm^2/ms.  k = 28.4: PAPER.md:96.
  static const double fhn[5] = {1.0, 1.5, 0.05, 1.5, -0.1};
  static const double karma[9] = {0.0011, 2.5, 250.0, 3.0, 1.0, 1.5415, 1.0, 6.0, 28.4};
  static const double bocf[30] = {1.171e-3, 28.4,   0.0,    1.55,   0.3,    0.13,    0.006,  0.006,
                                  60.0,     1150.0, 1.4506, 60.0,   15.0,   65.0,    0.03,   200.0,
                                  0.11,     400.0,  6.0,    30.0181, 0.9957, 2.0458, 0.65,   2.7342,
                                  16.0,     2.0994, 0.9087, 1.8875, 0.07,   0.94};
  const double* src = model == CARDIAC_FHN ? fhn : (model == CARDIAC_KARMA ? karma : bocf);
  std::memcpy(p, src, sizeof(double) * n);
  return CARDIAC_OK;
}

cardiac_ctx* cardiac_create3d(int model, int nx, int ny, int nz, double dx, double dt, int scheme, int batch) {
  auto bad = [](const std::string& m) -> cardiac_ctx* { g_create_error = m; return nullptr; };
  g_create_error.clear();
  const int nv = cardiac_num_fields(model);
  if (nv < 0) return bad("unknown model");
  const int stencil = scheme & 0xff, integ = (scheme >> 8) & 0xff, bc = (scheme >> 16) & 0xff,
            variant = (scheme >> 24) & 0xff;
  if (scheme < 0 || stencil > S_BOX9) return bad("unknown stencil bits");
  if (integ > I_IMPLICIT_EULER) return bad("unknown integrator bits");
  if (bc > B_PERIODIC) return bad("unknown boundary bits");
  if (variant > V_TANHFREE) return bad("unknown variant bits");
  if (integ >= I_RUSH_LARSEN && model != CARDIAC_BOCF)
    return bad("Rush-Larsen / implicit Euler are defined for the BOCF gates only");
  const int r = stencil_radius(stencil);
  if (nx < 2 * r + 1 || ny < 2 * r + 1) return bad("nx, ny must be >= 2*radius+1");
  if (nx > (1 << 20) || ny > (1 << 20) || (long long)((nx + 15) / 16 * 16) * ny >= (1LL << 31))
    return bad("grid too large (a plane must have fewer than 2^31 elements)");
  if (batch < 1 || batch > 65535) return bad("batch must be in [1, 65535]");
  if (nz != 1) {   // 3-D: the same per-axis stencil along z
    if (nz < 2 * r + 1) return bad("nz must be 1 (2-D) or >= 2*radius+1");
    if (stencil == S_BOX9) return bad("the 3x3 box stencil (Eq. 6) is defined in 2-D only");
    if ((long long)batch * nz > 65535) return bad("batch * nz must be <= 65535");
  }
  if (!(dx > 0.0) || !std::isfinite(dx)) return bad("dx must be finite and > 0");
  if (!(dt > 0.0) || !std::isfinite(dt)) return bad("dt must be finite and > 0");

  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return bad(std::string("no CUDA device: ") + cudaGetErrorString(e));
  cudaDeviceProp prop{};
  e = cudaGetDeviceProperties(&prop, dev);
  if (e != cudaSuccess) return bad(std::string("cudaGetDeviceProperties: ") + cudaGetErrorString(e));
  if (prop.major != 10)
    return bad("libcardiac is built for sm_100a (B200) only; found compute capability " +
               std::to_string(prop.major) + "." + std::to_string(prop.minor));

  cardiac_ctx* c = new (std::nothrow) cardiac_ctx();
  if (!c) return bad("out of host memory");
  Problem& pb = c->pb;
  pb.model = model; pb.stencil = stencil; pb.integrator = integ; pb.boundary = bc;
  pb.variant = variant; pb.nx = nx; pb.ny = ny; pb.nz = nz; pb.batch = batch; pb.nv = nv;
  pb.nd = model == CARDIAC_FHN ? 2 : 1; pb.radius = r;
  pb.pitch = (nx + 15) / 16 * 16;
  pb.zstride = pb.pitch * ny;
  pb.fstride = (long long)pb.zstride * nz;
  pb.bstride = pb.fstride * nv;
  pb.dx = dx; pb.dt = dt;
  c->scheme = scheme;
  c->nparams = cardiac_num_params(model);
  cardiac_default_params(model, pb.params, c->nparams);
  c->device = dev;
  c->nbuf = buffers_of(integ);
  c->plan_req = CARDIAC_PLAN_AUTO;
  c->plan = auto_plan(pb);
  c->plan_param = c->plan != CARDIAC_PLAN_FUSED ? 0 : (integ == I_EULER ? kEulerBlock : fused_window_auto(pb));
  e = cudaStreamCreateWithFlags(&c->cap_stream, cudaStreamNonBlocking);
  if (e != cudaSuccess) {
    delete c;
    return bad(std::string("cudaStreamCreate: ") + cudaGetErrorString(e));
  }
  return c;
}

cardiac_ctx* cardiac_create(int model, int nx, int ny, double dx, double dt, int scheme, int batch) {
  return cardiac_create3d(model, nx, ny, 1, dx, dt, scheme, batch);
}

int cardiac_set_params(cardiac_ctx* c, const double* p, int n) {
  if (!c) return CARDIAC_ERR_INVALID;
  if (!p || n != c->nparams) return fail(c, CARDIAC_ERR_INVALID, "wrong parameter count");
  for (int i = 0; i < n; ++i)
    if (!std::isfinite(p[i])) return fail(c, CARDIAC_ERR_INVALID, "non-finite parameter");
  if (c->pb.model == CARDIAC_KARMA) {
    double M = p[7];
    if (M != std::floor(M) || M < 1 || M > 16)
      return fail(c, CARDIAC_ERR_INVALID, "Karma M must be an integer in [1,16]");
  }
  std::memcpy(c->pb.params, p, sizeof(double) * n);
  drop_graphs(c);
  return CARDIAC_OK;
}

int cardiac_get_params(const cardiac_ctx* c, double* p, int n) {
  if (!c || !p || n != c->nparams) return CARDIAC_ERR_INVALID;
  std::memcpy(p, c->pb.params, sizeof(double) * n);
  return CARDIAC_OK;
}

int cardiac_set_stream(cardiac_ctx* c, void* cuda_stream) {
  if (!c) return CARDIAC_ERR_INVALID;
  c->stream = (cudaStream_t)cuda_stream;
  return CARDIAC_OK;
}

int cardiac_set_plan(cardiac_ctx* c, int plan, int param) {
  if (!c) return CARDIAC_ERR_INVALID;
  int resolved = plan, rparam = 0, fimpl = 0;
  if (param < 0) return fail(c, CARDIAC_ERR_INVALID, "plan parameter must be >= 0");
  const int integ = c->pb.integrator;
  const bool rk_like = integ == I_EULER || integ == I_HEUN || integ == I_RK4;
  if (plan == CARDIAC_PLAN_AUTO) resolved = auto_plan(c->pb);
  if (resolved == CARDIAC_PLAN_STAGE) {
    if (param < 0 || param > 2)
      return fail(c, CARDIAC_ERR_INVALID, "STAGE: parameter must be 0 (auto), 1 (direct) or 2 (TMA ring)");
    if (param == 2 && c->pb.nz > 1 && !stage_ring3d_supported(c->pb, K_SELF))
      return fail(c, CARDIAC_ERR_INVALID, "the TMA-ring stage kernels are not available for this 3-D context");
    rparam = param;
  } else if (c->pb.nz > 1) {
    return fail(c, CARDIAC_ERR_INVALID, "3-D contexts run plan STAGE only");
  } else if (resolved == CARDIAC_PLAN_FUSED) {
    if (!rk_like) return fail(c, CARDIAC_ERR_INVALID, "FUSED supports Euler, Heun and RK4 only");
    fimpl = param >> 4;
    param &= 15;
    if (fimpl < 0 || fimpl > 2) return fail(c, CARDIAC_ERR_INVALID, "FUSED: implementation (parameter / 16) must be 0, 1 or 2");
    if (integ == I_EULER) {
      rparam = param == 0 ? kEulerBlock : param;
      if (rparam != 1 && rparam != kEulerBlock)
        return fail(c, CARDIAC_ERR_INVALID, "FUSED + Euler: steps per launch must be 1 or 4");
    } else {
      if (param < 0 || param > 8 || param == 6 || (param >= 2 && c->pb.nv > 2) || (param >= 3 && integ != I_RK4))
        return fail(c, CARDIAC_ERR_INVALID,
                    "FUSED + Heun/RK4: parameter 0 (auto), 1 (80x48 window), 2 (48x40 window, 2-field models) "
                    "or 3 / 4 / 5 / 7 / 8 (64x56 / 64x48 / 56x48 / 64x56 on 896 threads / 64x32 on 1024 threads, 2-field models, RK4)");
      rparam = param == 0 ? fused_window_auto(c->pb) : param;
    }
  } else if (resolved == CARDIAC_PLAN_PAIR) {
    if (!rk_like) return fail(c, CARDIAC_ERR_INVALID, "PAIR supports Euler, Heun and RK4 only");
    if (param < 0 || param > 2)
      return fail(c, CARDIAC_ERR_INVALID, "PAIR: parameter must be 0 (auto), 1 (direct) or 2 (TMA-fed persistent CTAs)");
    if (param == 2 && !pair_tma_supported(c->pb))
      return fail(c, CARDIAC_ERR_INVALID, "PAIR: the TMA implementation is not available for this context");
    rparam = param;
  } else if (resolved == CARDIAC_PLAN_PERSISTENT) {
    if (!resident_supported(c->pb))
      return fail(c, CARDIAC_ERR_INVALID,
                  "PERSISTENT needs Euler/Heun/RK4 and a grid that fits one cluster: C x 4096 cells (4-field model: C x 2048), C = 16 CTAs for batches of up to 4 members, else 8");
    if (param != 0) return fail(c, CARDIAC_ERR_INVALID, "plan parameter must be 0");
  } else {
    return fail(c, CARDIAC_ERR_INVALID, "plan not available for this context");
  }
  c->plan_req = plan;
  c->plan = resolved;
  c->plan_param = rparam;
  if (fimpl == 2 && !fused_tma_supported(c->pb, integ == I_EULER ? 1 : rparam, integ == I_EULER ? rparam : 1))
    return fail(c, CARDIAC_ERR_INVALID, "FUSED: the TMA implementation does not support this context / window");
  c->fused_impl = fimpl;
  c->pb.stage_impl = resolved == CARDIAC_PLAN_STAGE ? rparam : 0;
  c->pb.pair_impl = resolved == CARDIAC_PLAN_PAIR ? rparam : 0;
  drop_graphs(c);
  return CARDIAC_OK;
}

int cardiac_get_plan(const cardiac_ctx* c) { return c ? c->plan : CARDIAC_ERR_INVALID; }

size_t cardiac_workspace_bytes(const cardiac_ctx* c) {
  if (!c) return 0;
  return buffer_doubles(c->pb) * sizeof(double) * c->nbuf;
}

int cardiac_bind_workspace(cardiac_ctx* c, void* dev_ptr, size_t bytes) {
  if (!c) return CARDIAC_ERR_INVALID;
  if (c->ws) return fail(c, CARDIAC_ERR_INVALID, "workspace already bound");
  if (!dev_ptr) return fail(c, CARDIAC_ERR_INVALID, "null workspace");
  if (bytes < cardiac_workspace_bytes(c) || ((size_t)dev_ptr & 255))
    return fail(c, CARDIAC_ERR_WORKSPACE, "workspace too small or not 256-byte aligned");
  c->ws = dev_ptr;
  c->ws_bytes = bytes;
  c->ws_owned = false;
  carve(c);
  return CARDIAC_OK;
}

int cardiac_set_state(cardiac_ctx* c, const double* src, int src_on_device) {
  if (!c) return CARDIAC_ERR_INVALID;
  if (!src) return fail(c, CARDIAC_ERR_INVALID, "null source");
  DeviceGuard guard(c->device);
  int rc = ensure_workspace(c);
  if (rc) return rc;
  const Problem& pb = c->pb;
  c->cur = 0;
  CK(cudaMemcpy2DAsync(c->buf[0], (size_t)pb.pitch * sizeof(double), src,
                       (size_t)pb.nx * sizeof(double), (size_t)pb.nx * sizeof(double),
                       (size_t)pb.ny * pb.nz * pb.nv * pb.batch,
                       src_on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, c->stream));
  if (!src_on_device) CK(cudaStreamSynchronize(c->stream));
  c->has_state = true;
  return CARDIAC_OK;
}

int cardiac_get_state(cardiac_ctx* c, double* dst, int dst_on_device) {
  if (!c) return CARDIAC_ERR_INVALID;
  if (!dst) return fail(c, CARDIAC_ERR_INVALID, "null destination");
  if (!c->has_state) return fail(c, CARDIAC_ERR_NOSTATE, "no state set");
  DeviceGuard guard(c->device);
  const Problem& pb = c->pb;
  CK(cudaMemcpy2DAsync(dst, (size_t)pb.nx * sizeof(double), c->buf[c->cur],
                       (size_t)pb.pitch * sizeof(double), (size_t)pb.nx * sizeof(double),
                       (size_t)pb.ny * pb.nz * pb.nv * pb.batch,
                       dst_on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost, c->stream));
  if (!dst_on_device) CK(cudaStreamSynchronize(c->stream));
  return CARDIAC_OK;
}

int cardiac_step(cardiac_ctx* c, long long nsteps) {
  if (!c) return CARDIAC_ERR_INVALID;
  if (nsteps < 0) return fail(c, CARDIAC_ERR_INVALID, "nsteps < 0");
  if (!c->has_state) return fail(c, CARDIAC_ERR_NOSTATE, "no state set");
  if (nsteps == 0) return CARDIAC_OK;
  DeviceGuard guard(c->device);
  if (c->plan == CARDIAC_PLAN_PERSISTENT) {   // one launch, in place, whatever nsteps
    ResidentLaunch rl{c->buf[c->cur], nsteps};
    cudaError_t e = launch_resident(c->pb, rl, c->stream);
    if (e != cudaSuccess) return fail_cuda(c, e, "resident launch");
    c->launches++;
    return CARDIAC_OK;
  }
  const int us = unit_steps(c);                                        // time steps per unit
  const int ul = c->plan == CARDIAC_PLAN_FUSED ? 1   // launches per unit
                 : (c->plan == CARDIAC_PLAN_PAIR ? (c->pb.integrator == I_RK4 ? 2 : 1) : stages_of(c->pb.integrator));
  int gunits = kGraphNodes / ul;
  if (gunits & 1) gunits++;  // even: ping-pong plans end on the parity they started on
  if (c->plan == CARDIAC_PLAN_PAIR) gunits = gunits / 6 * 6;   // ... and the rotation through 2 or 3 buffers
  const long long gsteps = (long long)gunits * us;
  long long left = nsteps;
  if (left >= gsteps) {
    if (c->graph_steps != gunits) drop_graphs(c);
    if (!c->graph[c->cur]) {
      int rc = build_graph(c, gunits);
      if (rc) return rc;
    }
    while (left >= gsteps) {
      CK(cudaGraphLaunch(c->graph[c->cur], c->stream));
      c->launches += (long long)gunits * ul;
      left -= gsteps;
    }
  }
  for (; left >= us; left -= us) {
    int rc = enqueue_unit(c, c->stream);
    if (rc) return rc;
  }
  for (; left > 0; --left) {  // fewer Euler steps than one temporal block
    int rc = enqueue_step(c, c->stream);
    if (rc) return rc;
  }
  return CARDIAC_OK;
}

int cardiac_get_jvp(cardiac_ctx* c, double eps, double* dst, int dst_on_device) {
  if (!c) return CARDIAC_ERR_INVALID;
  if (!dst) return fail(c, CARDIAC_ERR_INVALID, "null destination");
  if (!c->has_state) return fail(c, CARDIAC_ERR_NOSTATE, "no state set");
  if (c->pb.batch < 2) return fail(c, CARDIAC_ERR_INVALID, "JVP needs batch >= 2");
  if (!(eps != 0.0) || !std::isfinite(eps)) return fail(c, CARDIAC_ERR_INVALID, "bad eps");
  DeviceGuard guard(c->device);
  const Problem& pb = c->pb;
  if (dst_on_device) {
    cudaError_t e = launch_jvp(pb, c->buf[c->cur], eps, dst, c->stream);
    if (e != cudaSuccess) return fail_cuda(c, e, "jvp launch");
    c->launches++;
    return CARDIAC_OK;
  }
  const size_t bytes = (size_t)pb.nx * pb.ny * pb.nz * pb.nv * (pb.batch - 1) * sizeof(double);
  double* tmp = scratch_buffer(c);
  cudaError_t e = launch_jvp(pb, c->buf[c->cur], eps, tmp, c->stream);
  if (e == cudaSuccess) e = cudaMemcpyAsync(dst, tmp, bytes, cudaMemcpyDeviceToHost, c->stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
  if (e != cudaSuccess) return fail_cuda(c, e, "jvp");
  c->launches++;
  return CARDIAC_OK;
}

namespace {
int rows_copy(cardiac_ctx* c, int j0, int nrows, double* buf, int on_device, bool pack) {
  if (!c) return CARDIAC_ERR_INVALID;
  if (!buf) return fail(c, CARDIAC_ERR_INVALID, "null buffer");
  if (!c->has_state) return fail(c, CARDIAC_ERR_NOSTATE, "no state set");
  const Problem& pb = c->pb;
  if (j0 < 0 || nrows < 0 || (long long)j0 + nrows > (long long)pb.ny * pb.nz)
    return fail(c, CARDIAC_ERR_INVALID, "row range outside the grid");
  if (nrows == 0) return CARDIAC_OK;
  DeviceGuard guard(c->device);
  if (on_device) {
    cudaError_t e = launch_rows(pb, c->buf[c->cur], j0, nrows, buf, pack, c->stream);
    if (e != cudaSuccess) return fail_cuda(c, e, "rows launch");
    c->launches++;
    return CARDIAC_OK;
  }
  const size_t bytes = (size_t)pb.batch * pb.nv * nrows * pb.nx * sizeof(double);
  double* tmp = scratch_buffer(c);
  cudaError_t e = cudaSuccess;
  if (!pack) e = cudaMemcpyAsync(tmp, buf, bytes, cudaMemcpyHostToDevice, c->stream);
  if (e == cudaSuccess) e = launch_rows(pb, c->buf[c->cur], j0, nrows, tmp, pack, c->stream);
  if (e == cudaSuccess && pack) e = cudaMemcpyAsync(buf, tmp, bytes, cudaMemcpyDeviceToHost, c->stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
  if (e != cudaSuccess) return fail_cuda(c, e, "rows copy");
  c->launches++;
  return CARDIAC_OK;
}
}  // namespace

int cardiac_get_rows(cardiac_ctx* c, int j0, int nrows, double* dst, int dst_on_device) {
  return rows_copy(c, j0, nrows, dst, dst_on_device, true);
}

int cardiac_set_rows(cardiac_ctx* c, int j0, int nrows, const double* src, int src_on_device) {
  return rows_copy(c, j0, nrows, const_cast<double*>(src), src_on_device, false);
}

int cardiac_probe(cardiac_ctx* c, int what, const double* in_dev, double* out_dev, long long n) {
  if (!c) return CARDIAC_ERR_INVALID;
  if (!in_dev || !out_dev || n < 0) return fail(c, CARDIAC_ERR_INVALID, "bad probe arguments");
  if (what < CARDIAC_PROBE_EXP || what > CARDIAC_PROBE_REACTION)
    return fail(c, CARDIAC_ERR_INVALID, "unknown probe");
  DeviceGuard guard(c->device);
  cudaError_t e = launch_probe(c->pb, what, in_dev, out_dev, n, c->stream);
  if (e != cudaSuccess) return fail_cuda(c, e, "probe launch");
  c->launches++;
  return CARDIAC_OK;
}

long long cardiac_launch_count(const cardiac_ctx* c) { return c ? c->launches : 0; }

int cardiac_time_steps(cardiac_ctx* c, long long nsteps, int reps, float* ms_total) {
  if (!c) return CARDIAC_ERR_INVALID;
  if (!ms_total || reps < 1) return fail(c, CARDIAC_ERR_INVALID, "bad arguments");
  DeviceGuard guard(c->device);
  cudaEvent_t e0, e1;
  CK(cudaEventCreate(&e0));
  CK(cudaEventCreate(&e1));
  int rc = CARDIAC_OK;
  cudaError_t e = cudaEventRecord(e0, c->stream);
  for (int r = 0; r < reps && rc == CARDIAC_OK && e == cudaSuccess; ++r) rc = cardiac_step(c, nsteps);
  if (e == cudaSuccess) e = cudaEventRecord(e1, c->stream);
  if (e == cudaSuccess) e = cudaEventSynchronize(e1);
  if (e == cudaSuccess) e = cudaEventElapsedTime(ms_total, e0, e1);
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  if (rc) return rc;
  if (e != cudaSuccess) return fail_cuda(c, e, "timing");
  return CARDIAC_OK;
}

namespace {
int measure_dfma(cardiac_ctx* c, int iters, int reps, int int_per_dfma, double* dfma_per_s);
}
int cardiac_measure_fp64_peak(cardiac_ctx* c, int iters, int reps, double* dfma_per_s) {
  return measure_dfma(c, iters, reps, -1, dfma_per_s);
}
int cardiac_measure_fp64_issue(cardiac_ctx* c, int iters, int reps, int int_per_dfma, double* dfma_per_s) {
  if (c && int_per_dfma != 0 && int_per_dfma != 2 && int_per_dfma != 4)
    return fail(c, CARDIAC_ERR_INVALID, "int_per_dfma must be 0, 2 or 4");
  return measure_dfma(c, iters, reps, int_per_dfma, dfma_per_s);
}
namespace {
// int_per_dfma < 0: the 8-chain peak kernel; else the 4-chain kernel with that many integer instructions per DFMA
int measure_dfma(cardiac_ctx* c, int iters, int reps, int int_per_dfma, double* dfma_per_s) {
  if (!c) return CARDIAC_ERR_INVALID;
  if (!dfma_per_s || iters < 1 || reps < 1) return fail(c, CARDIAC_ERR_INVALID, "bad arguments");
  DeviceGuard guard(c->device);
  int sms = 0;
  CK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, c->device));
  const int blocks = sms * 4;   // 4 x 256 threads = 32 warps per SM, all resident (launch bounds)
  double* sink = nullptr;
  CK(cudaMalloc(&sink, (size_t)blocks * kDfmaThreads * sizeof(double)));
  cudaEvent_t e0 = nullptr, e1 = nullptr;
  cudaError_t e = cudaEventCreate(&e0);
  if (e == cudaSuccess) e = cudaEventCreate(&e1);
  float best = 0.f;
  for (int r = 0; r <= reps && e == cudaSuccess; ++r) {   // r = 0: warm-up
    e = cudaEventRecord(e0, c->stream);
    if (e == cudaSuccess)
      e = int_per_dfma < 0 ? launch_dfma_peak(sink, blocks, iters, c->stream)
                           : launch_dfma_mix(sink, blocks, iters, int_per_dfma, c->stream);
    if (e == cudaSuccess) e = cudaEventRecord(e1, c->stream);
    if (e == cudaSuccess) e = cudaEventSynchronize(e1);
    float ms = 0.f;
    if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
    if (r > 0 && (best == 0.f || ms < best)) best = ms;
    c->launches++;
  }
  if (e0) cudaEventDestroy(e0);
  if (e1) cudaEventDestroy(e1);
  cudaFree(sink);
  if (e != cudaSuccess) return fail_cuda(c, e, "fp64 peak");
  const double per_thread = int_per_dfma < 0 ? (double)kDfmaChains * kDfmaUnroll : (double)kDfmaMixChains * kDfmaMixUnroll;
  const double n = (double)blocks * kDfmaThreads * per_thread * (double)iters;
  *dfma_per_s = n / ((double)best * 1e-3);
  return CARDIAC_OK;
}
}  // namespace

const char* cardiac_last_error(const cardiac_ctx* c) {
  return c ? c->err.c_str() : g_create_error.c_str();
}

void cardiac_destroy(cardiac_ctx* c) {
  if (!c) return;
  DeviceGuard guard(c->device);
  drop_graphs(c);
  if (c->ws_owned && c->ws) cudaFree(c->ws);
  if (c->cap_stream) cudaStreamDestroy(c->cap_stream);
  delete c;
}

}  // extern "C"
