// stream_kernels.cu — plan STAGE, implementation RING: the same fused stencil + reaction + RK-stage
// update per substep as stage_kernels.cu, fed by a TMA ring.
//
// Why: ncu on the direct kernel (profiles/, r1 v3) shows the 4-field ionic model at ~50 % of BOTH
// the FP64 pipe and the issue slots, at any grid size — L2-resident 768^2 runs no faster than 2048^2.
// Every warp is a one-shot "load -> wait -> ~650 instructions -> store", and the compiler sinks the
// loads of the gates, of the stencil neighbours and of the RK operands next to their first use, so a
// warp sits through three to four exposed memory latencies (long-scoreboard = 60 % of all stall
// samples).  Here the operands of a tile are moved global -> shared by the TMA unit
// (cp.async.bulk.tensor, one elected producer thread, 2 to 5 box copies per tile) one or more tiles
// AHEAD of the warps that consume them; the consumers only ever wait on shared memory.
//
//   CTA     : 4 warps, one tile row each, a thread = 2 x-adjacent cells; thread 0 also issues the box
//             copies of the tile NSLOT-1 iterations ahead; persistent, tiles handed out round-robin
//             (tile = blockIdx.x + k gridDim.x), x fastest
//   tile    : 64 x 4 cells of one batch member
//   slot    : [n_d halo boxes 68 x (4+2r)] [gating fields 64 x 4] [y] [Y2] [Y3]   (as the kind needs)
//   ring    : NSLOT slots, full/empty mbarriers (the canonical TMA producer/consumer pipeline)
//   boundary: TMA zero-fills outside the grid; on rim tiles the consumers overwrite those ghost cells
//             with the mirrored / wrapped cell (PAPER.md:104 Fig. 1, :114) before the stencil runs
//
// The arithmetic per cell is the one of stage_kernels.cu (same Stencil<>, Model<>::reaction,
// combine<>), so both implementations give bitwise identical results.
#include <cuda_runtime.h>

#include <atomic>
#include <cstdint>
#include <cstring>
#include <mutex>
#include <vector>

#include "plans.h"
#include "stage.cuh"
#include "tma.cuh"

namespace cardiac {

namespace {

constexpr int TW = 64;            // tile width  (cells) = 2 per lane
constexpr int TH = 4;             // tile height (cells) = consumer warps
constexpr int HP = TW + 4;        // halo-box row pitch: 2 ghost columns each side keeps 16-byte alignment
constexpr int NCONS = 32 * TH;    // consumer threads
constexpr int NTHREADS = NCONS;

constexpr int align128(int bytes) { return (bytes + 127) / 128 * 128; }

template <class MD, int STENCIL, int KIND>
struct SlotLayout {
  static constexpr int NV = MD::NV, ND = MD::ND, NG = NV - ND;
  static constexpr int R = stencil_radius(STENCIL);
  static constexpr int HR = TH + 2 * R;
  static constexpr int HALO_BYTES = ND * HR * HP * 8;
  static constexpr int GATE_BYTES = NG * TH * TW * 8;
  static constexpr int FULL_BYTES = NV * TH * TW * 8;
  static constexpr int OFF_GATE = align128(HALO_BYTES);
  static constexpr int OFF_Y = OFF_GATE + align128(GATE_BYTES);
  static constexpr int OFF_A = OFF_Y + (KIND != K_SELF ? FULL_BYTES : 0);
  static constexpr int OFF_B = OFF_A + (KIND == K_RK4F ? FULL_BYTES : 0);
  static constexpr int SLOT_BYTES = OFF_B + (KIND == K_RK4F ? FULL_BYTES : 0);
  static constexpr unsigned TX_BYTES =
      HALO_BYTES + GATE_BYTES + (KIND != K_SELF ? FULL_BYTES : 0) + (KIND == K_RK4F ? 2 * FULL_BYTES : 0);
  // ring depth: 2 to 4 slots within ~31 KB per CTA, so that 7 CTAs (28 warps at <= 72 registers)
  // share an SM when the slot is small; the prefetch distance NSLOT-1 is counted in tile times, and
  // a tile of the models with large slots takes thousands of cycles
  static constexpr int NSLOT = SLOT_BYTES * 4 <= 31 * 1024 ? 4 : (SLOT_BYTES * 3 <= 32 * 1024 ? 3 : 2);
  static constexpr int SMEM_BYTES = NSLOT * SLOT_BYTES + 128;  // + the mbarriers
};

template <class MD>
struct RingArgs {
  StageArgs<MD> a;
  unsigned tiles_x, ntiles;   // ntiles < 2^31
  FastDiv per_member, per_row;
};
template <class MD>
CARDIAC_D TilePos tile_pos(const RingArgs<MD>& ra, unsigned t) {
  return tile_pos_of(t, ra.per_member, ra.per_row, ra.tiles_x, TW, TH);
}

CARDIAC_D void consumer_sync() { __syncthreads(); }

template <class MD, int STENCIL, int KIND>
__global__ void __launch_bounds__(NTHREADS)
    ring_stage_kernel(const __grid_constant__ RingArgs<MD> ra, const __grid_constant__ CUtensorMap tm_halo,
                      const __grid_constant__ CUtensorMap tm_gate, const __grid_constant__ CUtensorMap tm_y,
                      const __grid_constant__ CUtensorMap tm_A, const __grid_constant__ CUtensorMap tm_B) {
  using L = SlotLayout<MD, STENCIL, KIND>;
  constexpr int NV = MD::NV, ND = MD::ND, NG = L::NG, R = L::R, HR = L::HR, NSLOT = L::NSLOT;
  extern __shared__ __align__(1024) unsigned char ring_smem[];
  uint64_t* full = reinterpret_cast<uint64_t*>(ring_smem + NSLOT * L::SLOT_BYTES);
  uint64_t* empty = full + NSLOT;
  const StageArgs<MD>& a = ra.a;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const bool producer = threadIdx.x == 0;

  // the box copies of tile t into slot s (producer thread only)
  auto issue = [&](unsigned t, int s) {
    const TilePos tp = tile_pos(ra, t);
    unsigned char* slot = ring_smem + s * L::SLOT_BYTES;
    mbar_arrive_expect_tx(full + s, L::TX_BYTES);
    tma_load_4d(slot, &tm_halo, tp.x0 - 2, tp.y0 - R, 0, tp.bz, full + s);
    if (NG > 0) tma_load_4d(slot + L::OFF_GATE, &tm_gate, tp.x0, tp.y0, 0, tp.bz, full + s);
    if (KIND != K_SELF) tma_load_4d(slot + L::OFF_Y, &tm_y, tp.x0, tp.y0, 0, tp.bz, full + s);
    if (KIND == K_RK4F) {
      tma_load_4d(slot + L::OFF_A, &tm_A, tp.x0, tp.y0, 0, tp.bz, full + s);
      tma_load_4d(slot + L::OFF_B, &tm_B, tp.x0, tp.y0, 0, tp.bz, full + s);
    }
  };

  if (producer) {
#pragma unroll
    for (int s = 0; s < NSLOT; ++s) {
      mbar_init(full + s, 1);
      mbar_init(empty + s, TH);
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    // prologue: tiles 0 .. NSLOT-2 of this CTA into the fresh slots 0 .. NSLOT-2
    unsigned t = blockIdx.x;
#pragma unroll
    for (int s = 0; s < NSLOT - 1; ++s, t += gridDim.x)
      if (t < ra.ntiles) issue(t, s);
  }
  __syncthreads();

  const int nx = a.g.nx, ny = a.g.ny, pitch = a.g.pitch, bc = a.g.boundary;
  int s = 0;              // slot of the tile being consumed
  unsigned phase = 0;     // ... and the parity of its `full` phase
  int sp = NSLOT - 1;     // slot the producer refills next: the one consumed in the previous iteration
  unsigned pphase = 1;    // parity of its `empty` phase (a fresh mbarrier reads as "phase 1 complete")
  for (unsigned t = blockIdx.x; t < ra.ntiles; t += gridDim.x) {
    if (producer) {
      // tile t + (NSLOT-1) gridDim goes into the slot that tile t - gridDim has just left
      const unsigned long long tn = (unsigned long long)t + (unsigned long long)(NSLOT - 1) * gridDim.x;
      if (tn < ra.ntiles) {
        mbar_wait(empty + sp, pphase);
        issue((unsigned)tn, sp);
      }
    }
    if (++sp == NSLOT) { sp = 0; pphase ^= 1; }
    __syncwarp();

    const TilePos tp = tile_pos(ra, t);
    const int x0 = tp.x0, y0 = tp.y0, bz = tp.bz;
    unsigned char* slot = ring_smem + s * L::SLOT_BYTES;
    double* halo = reinterpret_cast<double*>(slot);
    mbar_wait(full + s, phase);

    // rim tile: the box reaches outside the grid (zero-filled by the TMA unit) — fill the ghost cells
    // within r of the grid from their mirror / wrapped image (Q3; one reflection is
    // enough because nx, ny >= 2r+1)
    const bool rim_x = x0 < R || x0 + TW + R > nx, rim_y = y0 < R || y0 + TH + R > ny;
    if (rim_x || rim_y) {
      const double* inb = a.in + (long long)bz * a.g.bstride;
      if (rim_x) {  // ghost columns -r..-1 and nx..nx+r-1, every box row whose image exists
        for (int e = threadIdx.x; e < ND * HR * 2 * R; e += NCONS) {
          const int q = e / (HR * 2 * R), rr = (e / (2 * R)) % HR, k = e % (2 * R);
          const int gx = k < R ? -1 - k : nx + (k - R), gy = y0 - R + rr;
          const int cc = gx - x0 + 2;
          if (cc >= 0 && cc < HP && gy >= -R && gy < ny + R)
            halo[(q * HR + rr) * HP + cc] =
                inb[q * a.g.fstride + (long long)bidx(gy, ny, bc) * pitch + bidx(gx, nx, bc)];
        }
      }
      if (rim_y) {  // ghost rows -r..-1 and ny..ny+r-1 over the columns inside the grid
        for (int e = threadIdx.x; e < ND * 2 * R * HP; e += NCONS) {
          const int q = e / (2 * R * HP), k = (e / HP) % (2 * R), cc = e % HP;
          const int gy = k < R ? -1 - k : ny + (k - R), gx = x0 - 2 + cc;
          const int rr = gy - y0 + R;
          if (rr >= 0 && rr < HR && gx >= 0 && gx < nx)
            halo[(q * HR + rr) * HP + cc] =
                inb[q * a.g.fstride + (long long)bidx(gy, ny, bc) * pitch + gx];
        }
      }
      consumer_sync();
    }

    const int gx = x0 + 2 * lane, gy = y0 + warp;
    if (gx < nx && gy < ny) {
      const int hc = (warp + R) * HP + 2 + 2 * lane;   // centre of the pair inside a halo box
      const int pc = warp * TW + 2 * lane;             // ... inside a plain box
      double2 zz[NV];
#pragma unroll
      for (int q = 0; q < ND; ++q) zz[q] = ld2(halo + q * HR * HP + hc);
      const double* gate = reinterpret_cast<const double*>(slot + L::OFF_GATE);
#pragma unroll
      for (int q = ND; q < NV; ++q) zz[q] = ld2(gate + (q - ND) * TH * TW + pc);

      double z0[NV], z1[NV], f0[NV], f1[NV];
#pragma unroll
      for (int q = 0; q < NV; ++q) { z0[q] = zz[q].x; z1[q] = zz[q].y; }
      MD::reaction(a.p, z0, f0);
      MD::reaction(a.p, z1, f1);
#pragma unroll
      for (int q = 0; q < ND; ++q) {
        double s0, s1;
        stencil_pair<STENCIL>(halo + q * HR * HP, (warp + R) * HP, 2 + 2 * lane, HP, zz[q], s0, s1);
        f0[q] = fma(a.lapw[q], s0, f0[q]);
        f1[q] = fma(a.lapw[q], s1, f1[q]);
      }
      const double* Ys = reinterpret_cast<const double*>(slot + L::OFF_Y);
      const double* As = reinterpret_cast<const double*>(slot + L::OFF_A);
      const double* Bs = reinterpret_cast<const double*>(slot + L::OFF_B);
      double* ob = a.out + (long long)bz * a.g.bstride + (long long)gy * pitch + gx;
#pragma unroll
      for (int q = 0; q < NV; ++q) {
        double2 yy = make_double2(0.0, 0.0), AA = yy, BB = yy;
        if (KIND != K_SELF) yy = ld2(Ys + q * TH * TW + pc);
        if (KIND == K_RK4F) { AA = ld2(As + q * TH * TW + pc); BB = ld2(Bs + q * TH * TW + pc); }
        const double r0 = combine<KIND>(a.w_y, a.w_in, a.w_A, a.w_B, a.w_f, yy.x, z0[q], AA.x, BB.x, f0[q]);
        const double r1 = combine<KIND>(a.w_y, a.w_in, a.w_A, a.w_B, a.w_f, yy.y, z1[q], AA.y, BB.y, f1[q]);
        if (gx + 1 < nx) st2(ob + q * a.g.fstride, r0, r1);
        else ob[q * a.g.fstride] = r0;
      }
    }
    // this warp is done with the slot (generic-proxy writes of the rim patch before the next TMA write)
    if (rim_x || rim_y) asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    __syncwarp();
    if (lane == 0) mbar_arrive(empty + s);
    if (++s == NSLOT) { s = 0; phase ^= 1; }
  }
}

template <class MD, int STENCIL, int KIND>
cudaError_t run_ring(const Problem& pb, const StageLaunch& st, cudaStream_t stream) {
  using L = SlotLayout<MD, STENCIL, KIND>;
  auto kern = ring_stage_kernel<MD, STENCIL, KIND>;
  // per instantiation and device: the shared-memory limit, and the size of the persistent grid
  static PerDeviceOnce configured;
  static std::atomic<int> grid_of[64];
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 0 || dev >= 64) return cudaErrorInvalidDevice;
  e = configured.run([&] {
    cudaError_t e2 = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, L::SMEM_BYTES);
    if (e2 != cudaSuccess) return e2;
    int sms = 0, occ = 0;
    if ((e2 = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess) return e2;
    if ((e2 = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, NTHREADS, L::SMEM_BYTES)) != cudaSuccess)
      return e2;
    if (occ < 1) return cudaErrorLaunchOutOfResources;
    grid_of[dev].store(sms * occ, std::memory_order_relaxed);
    return cudaSuccess;
  });
  if (e != cudaSuccess) return e;
  RingArgs<MD> ra;
  StageArgs<MD>& a = ra.a;
  a.in = st.in; a.y = st.y ? st.y : st.in; a.A = st.A ? st.A : st.in; a.B = st.B ? st.B : st.in;
  a.out = st.out;
  a.g.nx = pb.nx; a.g.ny = pb.ny; a.g.pitch = pb.pitch; a.g.boundary = pb.boundary;
  a.g.nz = 1; a.g.zstride = pb.zstride;
  a.g.fstride = pb.fstride; a.g.bstride = pb.bstride;
  a.w_y = st.w_y; a.w_in = st.w_in; a.w_A = st.w_A; a.w_B = st.w_B; a.w_f = st.w_f;
  a.dt = pb.dt;
  MD::derive(pb.params, a.p);
  for (int q = 0; q < MD::ND; ++q) a.lapw[q] = a.p.D[q] * stencil_norm(STENCIL) / (pb.dx * pb.dx);
  const long long tiles_x = (pb.nx + TW - 1) / TW, tiles_y = (pb.ny + TH - 1) / TH;
  const long long ntiles = tiles_x * tiles_y * pb.batch;
  if (ntiles >= (1LL << 31)) return cudaErrorInvalidValue;   // stage_ring_supported() said so
  ra.tiles_x = (unsigned)tiles_x;
  ra.ntiles = (unsigned)ntiles;
  ra.per_member = make_fastdiv((unsigned)(tiles_x * tiles_y));
  ra.per_row = make_fastdiv((unsigned)tiles_x);

  CUtensorMap tm_halo, tm_gate, tm_y, tm_A, tm_B;
  if ((e = tensor_map_4d(a.in, pb, MD::ND, HP, L::HR, &tm_halo)) != cudaSuccess) return e;
  tm_gate = tm_halo;
  if (L::NG > 0 &&
      (e = tensor_map_4d(a.in + MD::ND * pb.fstride, pb, L::NG, TW, TH, &tm_gate)) != cudaSuccess)
    return e;
  tm_y = tm_A = tm_B = tm_halo;
  if (KIND != K_SELF && (e = tensor_map_4d(a.y, pb, MD::NV, TW, TH, &tm_y)) != cudaSuccess) return e;
  if (KIND == K_RK4F) {
    if ((e = tensor_map_4d(a.A, pb, MD::NV, TW, TH, &tm_A)) != cudaSuccess) return e;
    if ((e = tensor_map_4d(a.B, pb, MD::NV, TW, TH, &tm_B)) != cudaSuccess) return e;
  }
  long long grid = grid_of[dev].load(std::memory_order_relaxed);
  if (grid > ra.ntiles) grid = ra.ntiles;
  kern<<<(unsigned)grid, NTHREADS, L::SMEM_BYTES, stream>>>(ra, tm_halo, tm_gate, tm_y, tm_A, tm_B);
  return cudaGetLastError();
}

template <class MD, int STENCIL>
cudaError_t ring_by_kind(const Problem& pb, const StageLaunch& st, cudaStream_t s) {
  switch (st.kind) {
    case K_SELF: return run_ring<MD, STENCIL, K_SELF>(pb, st, s);
    case K_BASE: return run_ring<MD, STENCIL, K_BASE>(pb, st, s);
    case K_RK4F: return run_ring<MD, STENCIL, K_RK4F>(pb, st, s);
  }
  return cudaErrorInvalidValue;
}

template <class MD>
cudaError_t ring_by_stencil(const Problem& pb, const StageLaunch& st, cudaStream_t s) {
  switch (pb.stencil) {
    case S_LAP5: return ring_by_kind<MD, S_LAP5>(pb, st, s);
    case S_LAP9X4: return ring_by_kind<MD, S_LAP9X4>(pb, st, s);
    case S_BOX9: return ring_by_kind<MD, S_BOX9>(pb, st, s);
  }
  return cudaErrorInvalidValue;
}

}  // namespace

// ------------------------------------------------------------------ host: tensor maps (declared in tma.cuh)
namespace {
using EncodeTiledFn = CUresult (*)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                   const cuuint64_t*, const cuuint32_t*, const cuuint32_t*,
                                   CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion,
                                   CUtensorMapFloatOOBfill);

EncodeTiledFn encoder() {
  static EncodeTiledFn fn = [] {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) != cudaSuccess ||
        q != cudaDriverEntryPointSuccess)
      p = nullptr;
    return reinterpret_cast<EncodeTiledFn>(p);
  }();
  return fn;
}

struct MapKey {
  const void* base;
  int nx, ny, nz, nf, batch, pitch, bw, bh;   // nz = 0: the 4-D view of a 2-D grid
  long long zstride, fstride, bstride;
  bool operator==(const MapKey& o) const { return std::memcmp(this, &o, sizeof(MapKey)) == 0; }
};
struct MapEntry {
  MapKey key;
  CUtensorMap map;
};

}  // namespace

// 4-D view (x, y, field, batch member) of `nf` fields starting at `base`; box = bw x bh x nf x 1
cudaError_t tensor_map_4d(const double* base, const Problem& pb, int nf, int bw, int bh, CUtensorMap* out) {
  static std::mutex mu;
  static std::vector<MapEntry> cache;
  MapKey k;
  std::memset(&k, 0, sizeof(k));
  k.base = base; k.nx = pb.nx; k.ny = pb.ny; k.nf = nf; k.batch = pb.batch; k.pitch = pb.pitch;
  k.bw = bw; k.bh = bh; k.fstride = pb.fstride; k.bstride = pb.bstride;
  std::lock_guard<std::mutex> lock(mu);
  for (const MapEntry& e : cache)
    if (e.key == k) { *out = e.map; return cudaSuccess; }
  EncodeTiledFn enc = encoder();
  if (!enc) return cudaErrorNotSupported;
  const cuuint64_t gdim[4] = {(cuuint64_t)pb.nx, (cuuint64_t)pb.ny, (cuuint64_t)nf, (cuuint64_t)pb.batch};
  const cuuint64_t gstr[3] = {(cuuint64_t)pb.pitch * 8, (cuuint64_t)pb.fstride * 8, (cuuint64_t)pb.bstride * 8};
  const cuuint32_t box[4] = {(cuuint32_t)bw, (cuuint32_t)bh, (cuuint32_t)nf, 1};
  const cuuint32_t estr[4] = {1, 1, 1, 1};
  CUtensorMap m;
  CUresult r = enc(&m, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 4, const_cast<double*>(base), gdim, gstr, box, estr,
                   CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                   CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) return cudaErrorInvalidValue;
  if (cache.size() >= 256) cache.clear();
  cache.push_back({k, m});
  *out = m;
  return cudaSuccess;
}

// 5-D view (x, y, z, field, batch member) of a 3-D grid; box = bw x bh x 1 x nf x 1 (one plane)
cudaError_t tensor_map_5d(const double* base, const Problem& pb, int nf, int bw, int bh, CUtensorMap* out) {
  static std::mutex mu;
  static std::vector<MapEntry> cache;
  MapKey k;
  std::memset(&k, 0, sizeof(k));
  k.base = base; k.nx = pb.nx; k.ny = pb.ny; k.nz = pb.nz; k.nf = nf; k.batch = pb.batch; k.pitch = pb.pitch;
  k.bw = bw; k.bh = bh; k.zstride = pb.zstride; k.fstride = pb.fstride; k.bstride = pb.bstride;
  std::lock_guard<std::mutex> lock(mu);
  for (const MapEntry& e : cache)
    if (e.key == k) { *out = e.map; return cudaSuccess; }
  EncodeTiledFn enc = encoder();
  if (!enc) return cudaErrorNotSupported;
  const cuuint64_t gdim[5] = {(cuuint64_t)pb.nx, (cuuint64_t)pb.ny, (cuuint64_t)pb.nz, (cuuint64_t)nf, (cuuint64_t)pb.batch};
  const cuuint64_t gstr[4] = {(cuuint64_t)pb.pitch * 8, (cuuint64_t)pb.zstride * 8, (cuuint64_t)pb.fstride * 8,
                              (cuuint64_t)pb.bstride * 8};
  const cuuint32_t box[5] = {(cuuint32_t)bw, (cuuint32_t)bh, 1, (cuuint32_t)nf, 1};
  const cuuint32_t estr[5] = {1, 1, 1, 1, 1};
  CUtensorMap m;
  CUresult r = enc(&m, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 5, const_cast<double*>(base), gdim, gstr, box, estr,
                   CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                   CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) return cudaErrorInvalidValue;
  if (cache.size() >= 256) cache.clear();
  cache.push_back({k, m});
  *out = m;
  return cudaSuccess;
}

bool tma_available() { return encoder() != nullptr; }

bool stage_ring_supported(const Problem& pb, int kind) {
  if (kind != K_SELF && kind != K_BASE && kind != K_RK4F) return false;
  if (pb.nz > 1) return false;   // the ring tiles are 2-D
  // tensor-map limits: strides are multiples of 16 bytes by construction (pitch % 16 == 0)
  const long long ntiles = (long long)((pb.nx + TW - 1) / TW) * ((pb.ny + TH - 1) / TH) * pb.batch;
  return ntiles < (1LL << 31) && tma_available();
}

bool fused_tma_supported(const Problem& pb, int window, int ksteps) {
  if (pb.nz > 1 || pb.nv > 2 || pb.integrator > I_RK4 || window < 1 || window > 7 || (window >= 4 && window <= 6)) return false;
  if (pb.integrator == I_EULER && ksteps != kEulerBlock) return false;
  if (pb.integrator != I_RK4 && window >= 3) return false;
  const int ns = pb.integrator == I_RK4 ? 4 : (pb.integrator == I_HEUN ? 2 : ksteps);
  const int H = pb.radius * ns;
  int tw, th;
  fused_tile_of(pb.integrator == I_EULER ? 1 : window, H, tw, th);
  if (tw <= 0 || th <= 0 || pb.nx <= H + tw || pb.ny <= H + th) return false;   // one reflection maps every window index
  const long long ntiles = (long long)((pb.nx + tw - 1) / tw) * ((pb.ny + th - 1) / th) * pb.batch;
  return ntiles < (1LL << 31) && tma_available();
}

bool pair_tma_supported(const Problem& pb) {
  if (pb.nz > 1 || pb.integrator > I_RK4) return false;
  const long long ntiles = (long long)((pb.nx + 63) / 64) * ((pb.ny + 23) / 24) * pb.batch;
  return ntiles < (1LL << 31) && tma_available();
}

cudaError_t launch_stage_ring(const Problem& pb, const StageLaunch& st, cudaStream_t stream) {
  if (pb.model == M_FHN) return ring_by_stencil<Model<M_FHN, V_PAPER>>(pb, st, stream);
  if (pb.model == M_KARMA)
    return pb.variant == V_TANHFREE ? ring_by_stencil<Model<M_KARMA, V_TANHFREE>>(pb, st, stream)
                                    : ring_by_stencil<Model<M_KARMA, V_PAPER>>(pb, st, stream);
  if (pb.model == M_BOCF)
    return pb.variant == V_TANHFREE ? ring_by_stencil<Model<M_BOCF, V_TANHFREE>>(pb, st, stream)
                                    : ring_by_stencil<Model<M_BOCF, V_PAPER>>(pb, st, stream);
  return cudaErrorInvalidValue;
}

}  // namespace cardiac
