/*
 * cardiac_static.h — ONE entry point of libcardiac.so that allocates nothing.
 *
 * Why: some callers cannot call cudaMalloc — code under CUDA-graph capture, tight serving loops,
 * harnesses that forbid it.  The context API of cardiac.h keeps the stage values of a time step
 * (the intermediate values Y2, Y3, Y4 of a Runge-Kutta step; one
 * kernel per substep, each reading what the previous one wrote) in a workspace that is either
 * cudaMalloc'ed on first use or bound by the caller.  cardiac_step_static runs the same
 * stage-synchronous kernels (plan STAGE, DIRECT implementation: the same instruction sequence per
 * cell, bitwise the same results) with those stage buffers in a file-scope
 *     static __device__ __align__(256) array of CARDIAC_STATIC_SCRATCH_BYTES bytes
 * inside the library.  No cudaMalloc / cudaFree / allocating library routine and no host heap
 * allocation is made by the call; every GPU that loads the library holds the array until the
 * process exits.
 *
 * Limits and rules
 *   - 2-D grids only.  The call needs  n_buf x batch x n_v x ny x ceil16(nx) x 8  bytes of scratch
 *     (n_buf = 4 for RK4, 2 for every other integrator; ceil16 = nx rounded up to a multiple of 16)
 *     and is rejected with CARDIAC_ERR_WORKSPACE and a message naming both numbers when that
 *     exceeds CARDIAC_STATIC_SCRATCH_BYTES (32 MiB: e.g. BOCF RK4 up to 512 x 512, FHN / Karma RK4
 *     up to 720 x 720, Euler twice the cells).
 *   - Every call on a device shares that device's array, which keeps the last call's contents.
 *     Nothing in it has to start at zero: a call copies `in` over the state buffer first and
 *     every stage buffer is written (whole grid) by the substep before the one that reads it;
 *     the padding columns nx .. ceil16(nx)-1 are never read into a stored result.
 *   - Calls that overlap on the GPU (different streams, or the same stream from two host threads
 *     interleaving) RACE on the array: serialise them.  Calls on one stream are ordered.
 *   - Asynchronous like cardiac_step: everything is enqueued on `cuda_stream` (NULL = the legacy
 *     default stream) and the call returns without synchronising.  `in_dev` and `out_dev` are
 *     DEVICE pointers on the current device to dense states [batch][n_v][ny][nx] (cardiac.h
 *     conventions), owned by the caller; they may be the same buffer.
 *   - model, scheme, dx, dt, params / nparams: as cardiac_create and cardiac_set_params
 *     (params = NULL: the defaults of cardiac_default_params).  nsteps >= 0.
 *   - errbuf (may be NULL) receives the error text, at most errbuf_len bytes including the NUL.
 *   - Returns CARDIAC_OK or a negative CARDIAC_ERR_* code; on an error nothing was enqueued
 *     unless the code is CARDIAC_ERR_CUDA (a launch failed part-way: `out_dev` is undefined).
 */
#ifndef CARDIAC_STATIC_H
#define CARDIAC_STATIC_H

#include "cardiac.h"

#ifdef __cplusplus
extern "C" {
#endif

#define CARDIAC_STATIC_SCRATCH_BYTES 33554432 /* 32 MiB per GPU that loads the library */

int cardiac_step_static(int model, int scheme, int nx, int ny, int batch, double dx, double dt,
                        const double* params, int nparams, const double* in_dev, double* out_dev,
                        long long nsteps, void* cuda_stream, char* errbuf, int errbuf_len);

#ifdef __cplusplus
}
#endif
#endif /* CARDIAC_STATIC_H */
