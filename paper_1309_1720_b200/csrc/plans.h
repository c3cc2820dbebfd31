// plans.h — host-side interface between the C-ABI (api.cu) and the kernel files.  Plain structs,
// no templates: each *_kernels.cu instantiates its kernels and exports one launcher.
#pragma once
#include <cuda_runtime.h>

namespace cardiac {

struct Problem {
  int model, stencil, integrator, boundary, variant;
  int nx, ny, batch, nv, nd, radius;
  int pitch;            // doubles per row
  long long fstride;    // doubles per field
  long long bstride;    // doubles per batch member
  double dx, dt;
  double params[32];    // public parameter block (include/cardiac.h)
  int stage_impl;       // plan STAGE: 0 = pick by size, 1 = DIRECT (stage_kernels.cu), 2 = RING (stream_kernels.cu)
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

// jvp: J[b-1] = (Z[b] - Z[0]) / eps, pitched state -> dense output
cudaError_t launch_jvp(const Problem& pb, const double* state, double eps, double* dst_dense,
                       cudaStream_t stream);

// tile_kernels_*.cu: plan FUSED — all substeps of one time step (ksteps = 1), or ksteps forward-Euler
// steps, in one launch on overlapped tiles (tile.cuh).  in != out.
constexpr int kEulerBlock = 4;  // Euler steps per launch when temporally blocked
struct TileLaunch {
  const double* in;
  double* out;
  int ksteps;
};
cudaError_t launch_fused_fhn(const Problem& pb, const TileLaunch& tl, cudaStream_t stream);
cudaError_t launch_fused_karma(const Problem& pb, const TileLaunch& tl, cudaStream_t stream);
cudaError_t launch_fused_bocf(const Problem& pb, const TileLaunch& tl, cudaStream_t stream);
inline cudaError_t launch_fused(const Problem& pb, const TileLaunch& tl, cudaStream_t stream) {
  return pb.model == 0 ? launch_fused_fhn(pb, tl, stream)
                       : (pb.model == 1 ? launch_fused_karma(pb, tl, stream)
                                        : launch_fused_bocf(pb, tl, stream));
}

// probe_kernels.cu: diagnostic evaluation of the device math / reactions on sample points
enum { PROBE_EXP = 0, PROBE_RCP = 1, PROBE_HK = 2, PROBE_REACTION = 3 };
cudaError_t launch_probe(const Problem& pb, int what, const double* in, double* out, long long n,
                         cudaStream_t stream);

}  // namespace cardiac
