// static_step.cu — cardiac_step_static (include/cardiac_static.h): time steps of plan STAGE whose stage buffers
// live in a file-scope __device__ array, for callers that must not allocate device memory.
//
// Nothing here is on the path of the context API (api.cu): the entry point builds its own Problem on the stack
// and sequences the existing DIRECT stage kernels (launch_stage, stage_kernels.cu) over buffers carved out of
// g_static_scratch.  No arithmetic of the method lives in this file.
#include <cuda_runtime.h>

#include <atomic>
#include <cmath>
#include <cstdarg>
#include <cstdio>

#include "../../include/cardiac_static.h"
#include "plans.h"
#include "stage.cuh"

using namespace cardiac;

namespace {

constexpr size_t kScratchDoubles = CARDIAC_STATIC_SCRATCH_BYTES / sizeof(double);

// The scratch.  In HOST code this name is only a handle for cudaGetSymbolAddress — not a device address.
static __device__ __align__(256) double g_static_scratch[kScratchDoubles];

// Device address of g_static_scratch on device d, looked up once per device with that device current
// (a benign race: two threads may both look it up and store the same value).
constexpr int kMaxDevices = 64;
std::atomic<double*> g_scratch_ptr[kMaxDevices];

int failf(char* errbuf, int errbuf_len, int code, const char* fmt, ...) {
  if (errbuf && errbuf_len > 0) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(errbuf, (size_t)errbuf_len, fmt, ap);
    va_end(ap);
  }
  return code;
}

cudaError_t scratch_address(double** out) {
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev >= 0 && dev < kMaxDevices) {
    double* p = g_scratch_ptr[dev].load(std::memory_order_acquire);
    if (p) { *out = p; return cudaSuccess; }
  }
  double* p = nullptr;
  e = cudaGetSymbolAddress((void**)&p, g_static_scratch);
  if (e != cudaSuccess) return e;
  if (!p) return cudaErrorInvalidSymbol;
  if (dev >= 0 && dev < kMaxDevices) g_scratch_ptr[dev].store(p, std::memory_order_release);
  *out = p;
  return cudaSuccess;
}

}  // namespace

extern "C" int cardiac_step_static(int model, int scheme, int nx, int ny, int batch, double dx, double dt,
                                   const double* params, int nparams, const double* in_dev, double* out_dev,
                                   long long nsteps, void* cuda_stream, char* errbuf, int errbuf_len) {
  auto bad = [&](const char* m) { return failf(errbuf, errbuf_len, CARDIAC_ERR_INVALID, "%s", m); };
  if (errbuf && errbuf_len > 0) errbuf[0] = 0;
  // ---- validation: the rules of cardiac_create / cardiac_set_params (api.cu), 2-D
  const int nv = cardiac_num_fields(model);
  if (nv < 0) return bad("unknown model");
  const int stencil = scheme & 0xff, integ = (scheme >> 8) & 0xff, bc = (scheme >> 16) & 0xff,
            variant = (scheme >> 24) & 0xff;
  if (scheme < 0 || stencil > S_BOX9) return bad("unknown stencil bits");
  if (integ > I_IMPLICIT_EULER) return bad("unknown integrator bits");
  if (bc > B_PERIODIC) return bad("unknown boundary bits");
  if (variant > 1) return bad("unknown variant bits");
  if (integ >= I_RUSH_LARSEN && model != CARDIAC_BOCF)
    return bad("Rush-Larsen / implicit Euler are defined for the BOCF gates only");
  const int r = stencil_radius(stencil);
  if (nx < 2 * r + 1 || ny < 2 * r + 1) return bad("nx, ny must be >= 2*radius+1");
  if (nx > (1 << 20) || ny > (1 << 20)) return bad("grid too large");
  if (batch < 1 || batch > 65535) return bad("batch must be in [1, 65535]");
  if (!(dx > 0.0) || !std::isfinite(dx)) return bad("dx must be finite and > 0");
  if (!(dt > 0.0) || !std::isfinite(dt)) return bad("dt must be finite and > 0");
  if (nsteps < 0) return bad("nsteps must be >= 0");
  if (!in_dev || !out_dev) return bad("null state pointer");

  Problem pb{};
  pb.model = model; pb.stencil = stencil; pb.integrator = integ; pb.boundary = bc; pb.variant = variant;
  pb.nx = nx; pb.ny = ny; pb.nz = 1; pb.batch = batch; pb.nv = nv;
  pb.nd = model == CARDIAC_FHN ? 2 : 1; pb.radius = r;
  pb.pitch = (nx + 15) / 16 * 16;
  pb.dx = dx; pb.dt = dt;
  pb.stage_impl = 1;   // DIRECT stage kernels: no tensor maps, nothing cached per buffer address
  pb.pair_impl = 0;
  const int np = cardiac_num_params(model);
  if (params) {
    if (nparams != np) return bad("wrong parameter count");
    for (int i = 0; i < np; ++i)
      if (!std::isfinite(params[i])) return bad("non-finite parameter");
    if (model == CARDIAC_KARMA) {
      const double M = params[7];
      if (M != std::floor(M) || M < 1 || M > 16) return bad("Karma M must be an integer in [1,16]");
    }
    for (int i = 0; i < np; ++i) pb.params[i] = params[i];
  } else {
    cardiac_default_params(model, pb.params, np);
  }

  // ---- the scratch: n_buf pitched state buffers
  const int nbuf = integ == I_RK4 ? 4 : 2;
  const unsigned long long per_buf = (unsigned long long)pb.pitch * ny * nv * batch;
  const unsigned long long need = per_buf * nbuf * sizeof(double);
  if (need > (unsigned long long)CARDIAC_STATIC_SCRATCH_BYTES)
    return failf(errbuf, errbuf_len, CARDIAC_ERR_WORKSPACE,
                 "cardiac_step_static needs %llu bytes of scratch for this problem (%d buffers of %d x %d x %d x %d "
                 "doubles); the static array holds %llu (CARDIAC_STATIC_SCRATCH_BYTES) — use the context API",
                 need, nbuf, batch, nv, ny, pb.pitch, (unsigned long long)CARDIAC_STATIC_SCRATCH_BYTES);
  pb.zstride = pb.pitch * ny;
  pb.fstride = pb.zstride;
  pb.bstride = pb.fstride * nv;

  double* scratch = nullptr;
  cudaError_t e = scratch_address(&scratch);
  if (e != cudaSuccess)
    return failf(errbuf, errbuf_len, CARDIAC_ERR_CUDA, "cudaGetSymbolAddress(static scratch): %s", cudaGetErrorString(e));
  double* buf[4];
  for (int i = 0; i < nbuf; ++i) buf[i] = scratch + (size_t)i * per_buf;   // per_buf is a multiple of 16 doubles

  cudaStream_t s = (cudaStream_t)cuda_stream;
  auto cuda_fail = [&](cudaError_t err, const char* what) {
    return failf(errbuf, errbuf_len, CARDIAC_ERR_CUDA, "%s: %s", what, cudaGetErrorString(err));
  };
  const size_t rows = (size_t)batch * nv * ny;
  e = cudaMemcpy2DAsync(buf[0], (size_t)pb.pitch * sizeof(double), in_dev, (size_t)nx * sizeof(double),
                        (size_t)nx * sizeof(double), rows, cudaMemcpyDeviceToDevice, s);
  if (e != cudaSuccess) return cuda_fail(e, "copy in");

  // ---- the launch sequence of plan STAGE (api.cu enqueue_step): same kinds, operands and weights
  StageLaunch st{};
  auto go = [&](int kind, const double* in, const double* y, const double* A, const double* B, double* out,
                double w_y, double w_in, double w_A, double w_B, double w_f) {
    st.kind = kind; st.in = in; st.y = y; st.A = A; st.B = B; st.out = out;
    st.w_y = w_y; st.w_in = w_in; st.w_A = w_A; st.w_B = w_B; st.w_f = w_f;
    return launch_stage(pb, st, s);
  };
  int cur = 0;
  for (long long n = 0; n < nsteps; ++n) {
    double* b0 = buf[cur];
    switch (integ) {
      case I_EULER:
      case I_RUSH_LARSEN:
      case I_IMPLICIT_EULER: {
        const int kind = integ == I_EULER ? K_SELF : (integ == I_RUSH_LARSEN ? K_RL : K_IE);
        e = go(kind, b0, nullptr, nullptr, nullptr, buf[cur ^ 1], 0, 0, 0, 0, dt);
        cur ^= 1;
        break;
      }
      case I_HEUN:
        e = go(K_SELF, b0, nullptr, nullptr, nullptr, buf[1], 0, 0, 0, 0, dt);
        if (e == cudaSuccess) e = go(K_BASE, buf[1], b0, nullptr, nullptr, b0, 0.5, 0.5, 0, 0, 0.5 * dt);
        break;
      default:   // I_RK4
        e = go(K_SELF, b0, nullptr, nullptr, nullptr, buf[1], 0, 0, 0, 0, 0.5 * dt);
        if (e == cudaSuccess) e = go(K_BASE, buf[1], b0, nullptr, nullptr, buf[2], 1.0, 0.0, 0, 0, 0.5 * dt);
        if (e == cudaSuccess) e = go(K_BASE, buf[2], b0, nullptr, nullptr, buf[3], 1.0, 0.0, 0, 0, dt);
        if (e == cudaSuccess)
          e = go(K_RK4F, buf[3], b0, buf[1], buf[2], b0, -1.0 / 3.0, 1.0 / 3.0, 1.0 / 3.0, 2.0 / 3.0, dt / 6.0);
        break;
    }
    if (e != cudaSuccess) return cuda_fail(e, "stage launch");
  }
  e = cudaMemcpy2DAsync(out_dev, (size_t)nx * sizeof(double), buf[cur], (size_t)pb.pitch * sizeof(double),
                        (size_t)nx * sizeof(double), rows, cudaMemcpyDeviceToDevice, s);
  if (e != cudaSuccess) return cuda_fail(e, "copy out");
  return CARDIAC_OK;
}
