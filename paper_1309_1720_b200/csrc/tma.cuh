// tma.cuh — what the TMA-fed kernels share (stream_kernels.cu: plan STAGE / RING; pairt.cuh: plan PAIR /
// TMA): PTX wrappers of the mbarrier / cp.async.bulk.tensor instructions, a division-free tile
// decomposition, and the host-side tensor-map cache (defined once, in stream_kernels.cu).
#pragma once
#include <cuda.h>   // CUtensorMap and its enums only; the encoder is fetched at run time (no -lcuda)
#include <cuda_runtime.h>

#include <cstdint>

#include "plans.h"
#include "stage.cuh"

namespace cardiac {

// n / d for n < 2^31 by one multiply-high and a shift (the round-up method of Granlund & Montgomery:
// m = ceil(2^(31 + ceil(log2 d)) / d)); the tile loop would otherwise spend ~150 instructions per
// tile on integer division, a third of the 4-field reaction itself
struct FastDiv {
  unsigned mul, shr, d;
};
inline FastDiv make_fastdiv(unsigned d) {
  FastDiv f;
  f.d = d;
  unsigned lg = 0;
  while ((1ull << lg) < d) ++lg;
  f.mul = (unsigned)(((1ull << (31 + lg)) + d - 1) / d);
  f.shr = lg == 0 ? 0 : lg - 1;
  return f;
}
CARDIAC_D unsigned fastdiv(unsigned n, const FastDiv& f) { return f.d == 1 ? n : __umulhi(n, f.mul) >> f.shr; }

// tile index -> (x0, y0, batch member) for tiles of tw x th cells handed out x fastest
struct TilePos {
  int x0, y0, bz;
};
CARDIAC_D TilePos tile_pos_of(unsigned t, const FastDiv& per_member, const FastDiv& per_row, unsigned tiles_x,
                              int tw, int th) {
  const unsigned bz = fastdiv(t, per_member), rem = t - bz * per_member.d;
  const unsigned ty = fastdiv(rem, per_row), tx = rem - ty * tiles_x;
  return {(int)tx * tw, (int)ty * th, (int)bz};
}
__host__ __device__ constexpr int tma_align128(int bytes) { return (bytes + 127) / 128 * 128; }

// ------------------------------------------------------------------ PTX wrappers
CARDIAC_D unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
CARDIAC_D void mbar_init(uint64_t* b, unsigned count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(b)), "r"(count) : "memory");
}
CARDIAC_D void mbar_arrive(uint64_t* b) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(b)) : "memory");
}
CARDIAC_D void mbar_arrive_expect_tx(uint64_t* b, unsigned bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(b)), "r"(bytes)
               : "memory");
}
CARDIAC_D void mbar_wait(uint64_t* b, unsigned parity) {
  unsigned ok;
  do {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(ok)
        : "r"(smem_u32(b)), "r"(parity)
        : "memory");
  } while (!ok);
}
CARDIAC_D void tma_load_4d(void* dst, const CUtensorMap* tm, int c0, int c1, int c2, int c3,
                           uint64_t* bar) {
  asm volatile(
      "cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes "
      "[%0], [%1, {%2, %3, %4, %5}], [%6];" ::"r"(smem_u32(dst)),
      "l"(reinterpret_cast<uint64_t>(tm)), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(smem_u32(bar))
      : "memory");
}
CARDIAC_D void tma_load_5d(void* dst, const CUtensorMap* tm, int c0, int c1, int c2, int c3, int c4,
                           uint64_t* bar) {
  asm volatile(
      "cp.async.bulk.tensor.5d.shared::cluster.global.mbarrier::complete_tx::bytes "
      "[%0], [%1, {%2, %3, %4, %5, %6}], [%7];" ::"r"(smem_u32(dst)),
      "l"(reinterpret_cast<uint64_t>(tm)), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(c4), "r"(smem_u32(bar))
      : "memory");
}
// ------------------------------------------------------------------ host
// 4-D view (x, y, field, batch member) of `nf` fields starting at `base` (a field of the pitched state
// buffers of `pb`), box = bw x bh x nf x 1; out-of-range elements are zero-filled.  Cached by value.
cudaError_t tensor_map_4d(const double* base, const Problem& pb, int nf, int bw, int bh, CUtensorMap* out);
// 5-D view (x, y, z, field, batch member) of a 3-D grid, box = bw x bh x 1 x nf x 1 (one plane)
cudaError_t tensor_map_5d(const double* base, const Problem& pb, int nf, int bw, int bh, CUtensorMap* out);
bool tma_available();   // the driver exports cuTensorMapEncodeTiled

}  // namespace cardiac
