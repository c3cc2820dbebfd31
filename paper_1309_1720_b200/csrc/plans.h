// plans.h — host-side interface between the C-ABI (api.cu) and the kernel files.  Plain structs,
// no templates: each *_kernels.cu instantiates its kernels and exports one launcher.
#pragma once
#include <cuda_runtime.h>

#include <atomic>

namespace cardiac {

// Function attributes (dynamic shared memory limit, non-portable cluster size) and occupancy are per
// DEVICE; a context captures the device it was created on (api.cu), so "done once" is kept per device:
// bit d of the mask = done on device d.  Safe from several host threads (setting an attribute twice is
// harmless; the bit is published after the call succeeded).
struct PerDeviceOnce {
  std::atomic<unsigned long long> mask{0};
  template <class F>
  cudaError_t run(F&& f) {
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= 64) return f();   // beyond the mask: configure every time
    const unsigned long long bit = 1ull << dev;
    if (mask.load(std::memory_order_acquire) & bit) return cudaSuccess;
    if ((e = f()) != cudaSuccess) return e;
    mask.fetch_or(bit, std::memory_order_release);
    return cudaSuccess;
  }
};

struct Problem {
  int model, stencil, integrator, boundary, variant;
  int nx, ny, nz, batch, nv, nd, radius;   // nz == 1: 2-D
  int pitch;            // doubles per row
  int zstride;          // doubles per plane (pitch * ny)
  long long fstride;    // doubles per field (zstride * nz)
  long long bstride;    // doubles per batch member
  double dx, dt;
  double params[32];    // public parameter block (include/cardiac.h)
  int stage_impl;       // plan STAGE: 0 = pick by size, 1 = DIRECT (stage_kernels.cu), 2 = RING (stream_kernels.cu)
  int pair_impl;        // plan PAIR: 0 = pick by size, 1 = DIRECT (pair.cuh), 2 = TMA (pairt.cuh)
};

// One stage launch of the STAGE plan (kind = K_* of stage.cuh).
struct StageLaunch {
  int kind;
  const double* in;
  const double* y;
  const double* A;
  const double* B;
  double* out;
  double w_y, w_in, w_A, w_B, w_f;
};

// stage_kernels.cu: fused stencil + reaction + RK-stage combine, one launch per substep.
cudaError_t launch_stage(const Problem& pb, const StageLaunch& st, cudaStream_t stream);

// stream_kernels.cu: the same stage update fed by a TMA ring (persistent CTAs); K_SELF/K_BASE/K_RK4F
bool stage_ring_supported(const Problem& pb, int kind);
cudaError_t launch_stage_ring(const Problem& pb, const StageLaunch& st, cudaStream_t stream);
constexpr long long kRingMinCells = 1 << 20;  // AUTO: below this the persistent grid has too few tiles per CTA
// stream3d_kernels.cu: ... for 3-D grids: persistent CTAs marching along z, planes of the diffusing fields by TMA
bool stage_ring3d_supported(const Problem& pb, int kind);
cudaError_t launch_stage_ring3d(const Problem& pb, const StageLaunch& st, cudaStream_t stream);

// jvp: J[b-1] = (Z[b] - Z[0]) / eps, pitched state -> dense output
cudaError_t launch_jvp(const Problem& pb, const double* state, double eps, double* dst_dense,
                       cudaStream_t stream);

// rows [j0, j0 + nrows) of the flattened (plane, row) index of every field and member: state -> dense
// [batch][n_v][nrows][nx] (pack) or back
cudaError_t launch_rows(const Problem& pb, double* state, int j0, int nrows, double* dense, bool pack,
                        cudaStream_t stream);

// tile_kernels_*.cu: plan FUSED — all substeps of one time step (ksteps = 1), or ksteps forward-Euler
// steps, in one launch on overlapped tiles (tile.cuh).  in != out.
constexpr int kEulerBlock = 4;  // Euler steps per launch when temporally blocked
struct TileLaunch {
  const double* in;
  double* out;
  int ksteps;
  int impl;    // 0 / 1 = fused_step_kernel (one CTA per tile), 2 = fused_tma_kernel (persistent CTAs fed by TMA, tilet.cuh)
  int window;  // Heun / RK4: 1 = 80 x 48 cells; two-field models also 2 = 48 x 40 (two CTAs per SM) and, RK4, 3 / 4 / 5 = 64 x 56 / 64 x 48 / 56 x 48
};
cudaError_t launch_fused_fhn(const Problem& pb, const TileLaunch& tl, cudaStream_t stream);
cudaError_t launch_fused_karma(const Problem& pb, const TileLaunch& tl, cudaStream_t stream);
cudaError_t launch_fused_bocf(const Problem& pb, const TileLaunch& tl, cudaStream_t stream);
inline cudaError_t launch_fused(const Problem& pb, const TileLaunch& tl, cudaStream_t stream) {
  return pb.model == 0 ? launch_fused_fhn(pb, tl, stream)
                       : (pb.model == 1 ? launch_fused_karma(pb, tl, stream)
                                        : launch_fused_bocf(pb, tl, stream));
}

// tilet_kernels_*.cu: plan FUSED, implementation TMA (two-field models; windows 1 - 3; Euler: blocked steps only)
cudaError_t launch_fusedt_fhn(const Problem& pb, const TileLaunch& tl, cudaStream_t stream);
cudaError_t launch_fusedt_karma(const Problem& pb, const TileLaunch& tl, cudaStream_t stream);
inline cudaError_t launch_fusedt(const Problem& pb, const TileLaunch& tl, cudaStream_t stream) {
  return pb.model == 0 ? launch_fusedt_fhn(pb, tl, stream)
                       : (pb.model == 1 ? launch_fusedt_karma(pb, tl, stream) : cudaErrorInvalidValue);
}
// window geometry (tile_dispatch.cuh FusedGeom) as the host needs it: output tile of window `win` at halo H
inline void fused_tile_of(int win, int H, int& tw, int& th) {
  const int ew = win == 2 ? 48 : (win == 3 || win == 4 || win == 7 || win == 8 ? 64 : (win == 5 ? 56 : 80));
  const int eh = win == 2 ? 40 : (win == 3 || win == 7 ? 56 : (win == 8 ? 32 : 48));
  tw = ew - 2 * H; th = eh - 2 * H;
}
bool fused_tma_supported(const Problem& pb, int window, int ksteps);
constexpr long long kFusedTMinTiles = 3 * 148;   // AUTO: every persistent CTA has several tiles to pipeline

// pair_kernels_*.cu: plan PAIR — two consecutive substeps per launch (pair.cuh): substep A (ka =
// K_SELF or K_BASE) on tile + ring into shared memory (and into `mid` when not null), substep B (kb)
// on the tile from shared memory into `out`.  out != in, out != y; out == A allowed.
struct PairLaunch {
  int ka, kb;
  const double* in;
  const double* y;
  const double* A;
  const double* B;
  double* mid;
  double* out;
  double a_wy, a_win, a_wf;
  double w_y, w_in, w_A, w_B, w_f;
};
constexpr long long kPairMinCellsRK4 = 9LL << 18, kPairMinCellsHeun = 12LL << 20;  // AUTO, 4-field model: 1536^2, 3584^2
cudaError_t launch_pair_fhn(const Problem& pb, const PairLaunch& pl, cudaStream_t stream);
cudaError_t launch_pair_karma(const Problem& pb, const PairLaunch& pl, cudaStream_t stream);
cudaError_t launch_pair_bocf(const Problem& pb, const PairLaunch& pl, cudaStream_t stream);
inline cudaError_t launch_pair(const Problem& pb, const PairLaunch& pl, cudaStream_t stream) {
  return pb.model == 0 ? launch_pair_fhn(pb, pl, stream)
                       : (pb.model == 1 ? launch_pair_karma(pb, pl, stream)
                                        : launch_pair_bocf(pb, pl, stream));
}

// pairt_kernels_*.cu: plan PAIR, implementation TMA (pairt.cuh) — the same two substeps per launch, persistent
// CTAs fed by TMA box copies.  RK4: launch 1 (ka = K_SELF, kb = K_BASE, out = Y3, out2 = P), launch 2
// (ka = K_BASE, kb = K_RK4F, in = Y3, y, P; out may be P's buffer).  out != in, out != y.
struct PairTLaunch {
  int ka, kb;
  const double* in;
  const double* y;
  const double* P;
  double* out;
  double* out2;
  double a_wy, a_win, a_wf;
  double w_y, w_in, w_f;
  double p_wy, p_wA, p_wB;
};
bool pair_tma_supported(const Problem& pb);   // 2-D, tensor maps available, fewer than 2^31 tiles
// AUTO picks the TMA implementation once every persistent CTA has several tiles to pipeline
constexpr long long kPairTMinTiles = 4 * 148;
// Below that a time step of the TMA pair kernels costs whole ROUNDS of one tile per persistent CTA (4-field model, round 2,
// LAP9X4: RK4 5.5 + 11.4 x rounds us, Heun 2.5 + 5.2 x rounds us), so it beats the launch-bound STAGE plan exactly where the
// last round is nearly full: 448^2 (133 tiles) 17.0 against 19.8 us per RK4 step, 640^2 (270) 28.4 / 30.7, 896^2 (532)
// 51.9 / 57.5 — and loses or ties at 512^2 (176 tiles: 28.4 / 21.7) and 768^2 (384: 39.9 / 39.6).
inline bool pair_tma_fills_rounds(long long tiles, int max_rounds) {
  const long long rounds = (tiles + 147) / 148;
  return tiles >= 120 && rounds <= max_rounds && tiles * 100 >= rounds * 148 * 88;
}
cudaError_t launch_pairt_fhn(const Problem& pb, const PairTLaunch& pl, cudaStream_t stream);
cudaError_t launch_pairt_karma(const Problem& pb, const PairTLaunch& pl, cudaStream_t stream);
cudaError_t launch_pairt_bocf(const Problem& pb, const PairTLaunch& pl, cudaStream_t stream);
inline cudaError_t launch_pairt(const Problem& pb, const PairTLaunch& pl, cudaStream_t stream) {
  return pb.model == 0 ? launch_pairt_fhn(pb, pl, stream)
                       : (pb.model == 1 ? launch_pairt_karma(pb, pl, stream)
                                        : launch_pairt_bocf(pb, pl, stream));
}

// resident_kernels_*.cu: plan PERSISTENT — one thread-block cluster of C <= 16 CTAs per batch member
// keeps the whole grid in (distributed) shared memory and advances all nsteps in ONE launch, in place
// (resident.cuh).  C CTAs of 512 threads x KP pairs: at most C x 4096 cells (2-field models) or
// C x 2048 cells (4-field model), C <= 16 for batches of up to 4 members (the non-portable cluster size)
// and <= 8 beyond; Euler / Heun / RK4.
struct ResidentLaunch {
  double* state;
  long long nsteps;
};
struct ResidentShape {
  int csize;   // CTAs per cluster (power of two, 0 = does not fit)
  int slab;    // rows per CTA
  size_t smem; // dynamic shared memory per CTA
};
constexpr size_t kResidentMaxSmem = 200 * 1024;   // per CTA
inline ResidentShape resident_shape(const Problem& pb) {
  ResidentShape rs{0, 0, 0};
  if (pb.integrator > 2 || pb.nz > 1) return rs;  // Euler, Heun, RK4; 2-D
  const long long npx = (pb.nx + 1) / 2, cap = 512LL * (pb.nv > 2 ? 2 : 4);
  const size_t sp = 2 * (size_t)npx + 4;
  const int cmax = pb.batch <= 4 ? 16 : 8;   // 16: non-portable size, at most one such cluster per GPC
  for (int c = 1; c <= cmax; c *= 2) {
    const int slab = (pb.ny + c - 1) / c;
    // two stage buffers framed by the ghost ring + the two mbarriers and the row-duty table of the ghost exchange
    const size_t smem = 2 * (size_t)pb.nd * sp * ((size_t)slab + 2 * pb.radius) * sizeof(double) + 16 + 256;
    if (c > 1 && slab < pb.radius) continue;   // the exchange reaches two CTAs up and down: slabs of at least r rows
    // fits, and one cell per thread where the grid is large enough to spread (a substep costs the
    // barrier plus the latency of one warp's instruction sequence, resident.cuh CPT)
    if (npx * slab <= cap && smem <= kResidentMaxSmem && (c == cmax || (pb.ny + 2 * c - 1) / (2 * c) < 4)) {
      rs.csize = c; rs.slab = slab; rs.smem = smem;
      return rs;
    }
  }
  return rs;
}
inline bool resident_supported(const Problem& pb) { return resident_shape(pb).csize > 0; }
// AUTO: measured on B200: a substep of the cluster-resident launch costs the ghost
// exchange (a remote store and the wait for the neighbours') and the latency of one warp's instruction
// sequence, which grows with the cells a CTA holds; against the per-step launches of FUSED / STAGE it wins up
// to (batch 1, 16 CTAs; round 2, push exchange, row-major cells) 192^2 for FHN Euler (1.37 against 1.69 us per
// step), 128^2 for FHN RK4 (4.5 / 5.0; 144^2: 5.5 / 5.0), 144^2 for Karma RK4 (5.0 / 5.6) and 128^2 for BOCF RK4
// (7.2 / 9.5) — expressed per CTA so that it carries
// over to the 8-CTA clusters of larger batches — and only while every cluster is resident at once (a GPC holds
// one cluster of 16, two of 8, four of 4: 17 members in clusters of 8 run as two waves, 8.0 against 6.0 us per
// FHN RK4 step at 64^2).
inline bool resident_preferred(const Problem& pb) {
  const ResidentShape rs = resident_shape(pb);
  if (rs.csize == 0) return false;
  const int max_clusters = rs.csize == 16 ? 4 : (rs.csize == 8 ? 16 : (rs.csize == 4 ? 32 : 144 / rs.csize));
  if (pb.batch > max_clusters) return false;
  const long long cells_per_cta = 2LL * ((pb.nx + 1) / 2) * rs.slab;
  // (against the best other plan, which for the 4-field model below 256^2 is the one-wave FUSED launch: RK4 128^2 7.2 / 9.5,
  // 160^2 12.0 / 9.5; Euler 128^2 1.9 / 2.2, 160^2 2.8 / 2.2; Heun 160^2 5.9 / 6.2 — and for Heun of the two-field models
  // 160^2 2.9 - 3.1 / 3.7 - 4.1, 192^2 a tie)
  const long long limit = pb.integrator == 1 ? 1700
                                             : (pb.nv > 2 ? 1100 : (pb.integrator == 0 ? 2400 : (pb.model == 0 ? 1100 : 1400)));
  return cells_per_cta <= limit;
}
cudaError_t launch_resident_fhn(const Problem& pb, const ResidentLaunch& rl, cudaStream_t stream);
cudaError_t launch_resident_karma(const Problem& pb, const ResidentLaunch& rl, cudaStream_t stream);
cudaError_t launch_resident_bocf(const Problem& pb, const ResidentLaunch& rl, cudaStream_t stream);
inline cudaError_t launch_resident(const Problem& pb, const ResidentLaunch& rl, cudaStream_t stream) {
  return pb.model == 0 ? launch_resident_fhn(pb, rl, stream)
                       : (pb.model == 1 ? launch_resident_karma(pb, rl, stream)
                                        : launch_resident_bocf(pb, rl, stream));
}

// probe_kernels.cu: diagnostic evaluation of the device math / reactions on sample points
enum { PROBE_EXP = 0, PROBE_RCP = 1, PROBE_HK = 2, PROBE_REACTION = 3 };
cudaError_t launch_probe(const Problem& pb, int what, const double* in, double* out, long long n,
                         cudaStream_t stream);


// FP64-pipe microbenchmark (cardiac_measure_fp64_peak): `blocks` CTAs of kDfmaThreads threads, each thread
// kDfmaChains independent chains of iters x kDfmaUnroll DFMAs; one double per thread is stored to `sink`
constexpr int kDfmaThreads = 256, kDfmaChains = 8, kDfmaUnroll = 64;
cudaError_t launch_dfma_peak(double* sink, int blocks, int iters, cudaStream_t stream);
// ... four chains of iters x kDfmaMixUnroll DFMAs per thread with int_per_dfma (0, 2 or 4) independent integer
// instructions in between (cardiac_measure_fp64_issue)
constexpr int kDfmaMixChains = 4, kDfmaMixUnroll = 16;
cudaError_t launch_dfma_mix(double* sink, int blocks, int iters, int int_per_dfma, cudaStream_t stream);

}  // namespace cardiac
