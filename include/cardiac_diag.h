/*
 * cardiac_diag.h — diagnostics of libcardiac.so: NOT part of the product boundary (include/cardiac.h).
 *
 * Entry points that tests and bench.py use to look inside the library: value-by-value evaluation of the
 * device-side math, launch counting, device-side timing, and the DFMA microbenchmark that measures the
 * FP64-pipe peak the roofline of the exp-heavy ionic model is reported against.
 * Same conventions as cardiac.h (int return = CARDIAC_OK or a negative CARDIAC_ERR_* code).
 */
#ifndef CARDIAC_DIAG_H
#define CARDIAC_DIAG_H

#include "cardiac.h"

#ifdef __cplusplus
extern "C" {
#endif

/* Evaluate device-side building blocks on n sample points held in device memory, enqueued on the
 * context stream.
 *   CARDIAC_PROBE_EXP      out[i] = the library's exp(in[i])            (used inside tanh)
 *   CARDIAC_PROBE_RCP      out[i] = the library's 1/in[i], in[i] > 0    (divisions)
 *   CARDIAC_PROBE_HK       out[i] = H_k(in[i]), k of the context's model
 *   CARDIAC_PROBE_REACTION in = [n][n_v] states, out = [n][n_v] reaction terms N[z] of the
 *                          context's model, variant and parameters */
enum { CARDIAC_PROBE_EXP = 0, CARDIAC_PROBE_RCP = 1, CARDIAC_PROBE_HK = 2, CARDIAC_PROBE_REACTION = 3 };
int cardiac_probe(cardiac_ctx*, int what, const double* in_dev, double* out_dev, long long n);

/* Total number of kernels this context has launched (graph nodes counted per replay). */
long long cardiac_launch_count(const cardiac_ctx*);

/* Run `nsteps` steps `reps` times back to back on the context stream and return, via CUDA events
 * recorded on that stream, the device time in milliseconds of the whole run in *ms_total
 * (synchronises the stream).  Used by bench.py for the live per-launch timing of the roofline. */
int cardiac_time_steps(cardiac_ctx*, long long nsteps, int reps, float* ms_total);

/* FP64-pipe peak of the context's device, measured: every SM runs 32 warps of 8 independent DFMA
 * chains each (registers only, no memory traffic) for `iters` x 64 DFMAs per chain; the launch is
 * timed with CUDA events on the context stream (synchronises it), best of `reps`.  *dfma_per_s =
 * thread-level DFMA instructions per second (x 2 = FLOP/s); the roofline of an ALU-bound path
 * (the paper's own peak estimate for its GPU) divides by this, not by a nominal figure.
 * iters >= 1, reps >= 1. */
int cardiac_measure_fp64_peak(cardiac_ctx*, int iters, int reps, double* dfma_per_s);

/* The same measurement with `int_per_dfma` (0, 2 or 4) independent integer instructions issued between the
 * DFMAs of four chains per thread: what an FP64 instruction costs a scheduler's ISSUE port.  On B200 the
 * rates come out as 1 / (2 + int_per_dfma) DFMA per cycle and scheduler — an FP64 instruction holds the port
 * for two cycles and nothing else issues meanwhile — so the bound of the exp-heavy ionic kernels
 * is 2 x (FP64 instructions) + (all other instructions), which bench.py reports beside
 * the FP64-pipe fraction. */
int cardiac_measure_fp64_issue(cardiac_ctx*, int iters, int reps, int int_per_dfma, double* dfma_per_s);

#ifdef __cplusplus
}
#endif
#endif /* CARDIAC_DIAG_H */
