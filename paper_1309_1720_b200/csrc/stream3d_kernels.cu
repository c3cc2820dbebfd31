// stream3d_kernels.cu — plan STAGE, implementation RING, for 3-D grids (DESIGN.md f4): the fused
// stencil + reaction + RK-stage update of stage_kernels.cu, marching along z with the planes of the diffusing
// fields arriving through a TMA ring.
//
// Why (ncu, round 2, FHN 13-point 256^3): the direct 3-D stage kernels spend 59-77 % of their stall samples on the
// long scoreboard — every pair issues 11 128-bit neighbour loads per diffusing field, five of them from other
// planes, and 28 warps per SM do not cover the L2 latency; the first three RK4 stages move 3.1-3.6 TB/s of the
// 6.5 TB/s copy bandwidth.  Round 1 tried marching along z with a REGISTER window (one exposed load latency per
// plane per warp: slower).  Here the planes are fetched ONCE per tile by the TMA unit, two planes ahead:
//
//   unit     an x-y tile of 64 x 8 cells x a chunk of up to 32 planes of one batch member; persistent CTAs (8 warps,
//            a warp = one tile row, a lane = an x-adjacent pair) take units round-robin
//   ring     2r+3 slots, each the halo box 68 x (8+2r) of every diffusing field of ONE plane
//            (cp.async.bulk.tensor.5d, full / empty mbarriers); the centre plane c needs the planes c-r .. c+r
//            resident: its own box for the in-plane stencil, the others' tile cells for the z arm; a plane beyond
//            the first / last one is the plane its index reflects or wraps to (the same box copy, another z)
//   operands the pointwise ones (gating fields, y, Y2, Y3 on the tile of the centre plane) come through a second,
//            shorter ring of box copies (a first version loaded them with 128-bit global loads at the top of an
//            iteration: one exposed DRAM latency per plane and warp, slower than the direct kernels)
//   boundary x / y: the TMA unit zero-fills outside the grid; rim tiles patch the ghost cells of each arriving
//            plane (patch_box, pairt.cuh)
//
// Same Stencil<>, StencilZ<>, Model<>::reaction, combine<> as stage_kernel<..., D3 = true>: bitwise identical results.
#include <atomic>

#include "pairt.cuh"   // patch_box
#include "plans.h"
#include "stage.cuh"
#include "tma.cuh"

namespace cardiac {

namespace {

constexpr int TW = 64, TH = 8, HP = TW + 4, NT = 32 * TH, ZC = 32;

template <class MD, int STENCIL>
struct Ring3D {
  static constexpr int ND = MD::ND;
  static constexpr int R = stencil_radius(STENCIL), NP = 2 * R + 1, HR = TH + 2 * R;
  static constexpr int FSZ = HR * HP;                       // doubles of one field of one plane
  static constexpr int SLOT_BYTES = tma_align128(ND * FSZ * 8);
  static constexpr unsigned TX_BYTES = ND * FSZ * 8;
  static constexpr int NSLOT = NP + 2;                      // two planes ahead of the deepest one in use
};
// the operand slot of one centre plane: [gating fields] [y] [Y2] [Y3] on the tile, as the kind needs
template <class MD, int STENCIL, int KIND>
struct Oper3D {
  using H = Ring3D<MD, STENCIL>;
  static constexpr int NV = MD::NV, ND = MD::ND, NG = NV - ND, TSZ = TH * TW;
  static constexpr int GATE_BYTES = NG * TSZ * 8, FULL_BYTES = NV * TSZ * 8;
  static constexpr int OFF_Y = tma_align128(GATE_BYTES);
  static constexpr int OFF_A = OFF_Y + (KIND != K_SELF ? FULL_BYTES : 0);
  static constexpr int OFF_B = OFF_A + (KIND == K_RK4F ? FULL_BYTES : 0);
  static constexpr int SLOT_BYTES = tma_align128(OFF_B + (KIND == K_RK4F ? FULL_BYTES : 0));
  static constexpr unsigned TX_BYTES = GATE_BYTES + (KIND != K_SELF ? FULL_BYTES : 0) + (KIND == K_RK4F ? 2 * FULL_BYTES : 0);
  static constexpr bool ANY = TX_BYTES > 0;
  static constexpr int NSLOT = !ANY ? 0 : (H::NSLOT * H::SLOT_BYTES + 3 * SLOT_BYTES <= 200 * 1024 ? 3 : 2);
  static constexpr int OFF_OPER = H::NSLOT * H::SLOT_BYTES, OFF_BAR = OFF_OPER + NSLOT * SLOT_BYTES;
  static constexpr int SMEM_BYTES = OFF_BAR + 256;
  static_assert(SMEM_BYTES <= 227 * 1024, "");
};

template <class MD>
struct Ring3DArgs {
  StageArgs<MD> a;
  unsigned tiles_x, nunits;
  int chunks;
  FastDiv per_member, per_chunk, per_row;
};

template <class MD, int STENCIL, int KIND>
__global__ void __launch_bounds__(NT, 2)
    ring3d_stage_kernel(const __grid_constant__ Ring3DArgs<MD> ra, const __grid_constant__ CUtensorMap tm_halo,
                        const __grid_constant__ CUtensorMap tm_gate, const __grid_constant__ CUtensorMap tm_y,
                        const __grid_constant__ CUtensorMap tm_A, const __grid_constant__ CUtensorMap tm_B) {
  using L = Ring3D<MD, STENCIL>;
  using P = Oper3D<MD, STENCIL, KIND>;
  constexpr int NV = MD::NV, ND = MD::ND, NG = NV - ND, R = L::R, HR = L::HR, FSZ = L::FSZ, NSLOT = L::NSLOT;
  constexpr int NSLOT_O = P::NSLOT, TSZ = P::TSZ;
  extern __shared__ __align__(1024) unsigned char r3_smem[];
  uint64_t* const full = reinterpret_cast<uint64_t*>(r3_smem + P::OFF_BAR);
  uint64_t* const empty = full + NSLOT;
  uint64_t* const full_o = empty + NSLOT;
  uint64_t* const empty_o = full_o + 3;
  const StageArgs<MD>& a = ra.a;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const bool producer = threadIdx.x == 0;
  const int nx = a.g.nx, ny = a.g.ny, nz = a.g.nz, pitch = a.g.pitch, bc = a.g.boundary;
  auto slot_of = [&](unsigned idx) { return reinterpret_cast<double*>(r3_smem + (idx % NSLOT) * L::SLOT_BYTES); };

  if (producer) {
#pragma unroll
    for (int s = 0; s < NSLOT; ++s) {
      mbar_init(full + s, 1);
      mbar_init(empty + s, TH);
    }
#pragma unroll
    for (int s = 0; s < 3; ++s) {
      mbar_init(full_o + s, 1);
      mbar_init(empty_o + s, TH);
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  }
  __syncthreads();

  unsigned base_idx = 0;   // ring index of plane 0 of the current unit (planes are numbered through all units)
  unsigned issued = 0;     // ring index of the next plane to request (producer)
  unsigned obase = 0, oissued = 0;   // the same for the operand ring (one entry per centre plane)
  for (unsigned u = blockIdx.x; u < ra.nunits; u += gridDim.x) {
    // unit -> (member, chunk, tile)
    const unsigned bz = fastdiv(u, ra.per_member), r1 = u - bz * ra.per_member.d;
    const unsigned ch = fastdiv(r1, ra.per_chunk), r2 = r1 - ch * ra.per_chunk.d;
    const unsigned ty = fastdiv(r2, ra.per_row), tx = r2 - ty * ra.tiles_x;
    const int x0 = (int)tx * TW, y0 = (int)ty * TH, z0 = (int)ch * ZC;
    const int zlen = min(ZC, nz - z0), nplanes = zlen + 2 * R;   // march planes m = 0 .. nplanes-1 = z0-R .. z0+zlen+R-1
    const long long mbase = (long long)bz * a.g.bstride;
    const bool rim = x0 < R || x0 + TW + R > nx || y0 < R || y0 + TH + R > ny;

    // request plane m of this unit (its slot was freed by the plane NSLOT requests earlier)
    auto request = [&](int m) {
      const unsigned idx = base_idx + (unsigned)m, s = idx % NSLOT, use = idx / NSLOT;
      mbar_wait(empty + s, (use & 1u) ^ 1u);   // a fresh mbarrier reads as "phase 1 complete"
      mbar_arrive_expect_tx(full + s, L::TX_BYTES);
      tma_load_5d(slot_of(idx), &tm_halo, x0 - 2, y0 - R, bidx(z0 - R + m, nz, bc), 0, (int)bz, full + s);
    };
    // all threads: plane m has arrived (and, on rim tiles, has its x / y ghost cells)
    auto arrived = [&](int m) {
      const unsigned idx = base_idx + (unsigned)m;
      mbar_wait(full + idx % NSLOT, (idx / NSLOT) & 1u);
      if (rim) {
        const int zz = bidx(z0 - R + m, nz, bc);
        patch_box<R>(slot_of(idx), ND, HP, HR, x0 - 2, y0 - R, a.in + mbase + (long long)zz * a.g.zstride, a.g,
                     threadIdx.x, NT);
      }
    };
    // the operand boxes of centre plane c of this unit
    auto request_op = [&](int c) {
      const unsigned idx = obase + (unsigned)c, s = idx % (NSLOT_O > 0 ? NSLOT_O : 1), use = idx / (NSLOT_O > 0 ? NSLOT_O : 1);
      unsigned char* slot = r3_smem + P::OFF_OPER + s * P::SLOT_BYTES;
      mbar_wait(empty_o + s, (use & 1u) ^ 1u);
      mbar_arrive_expect_tx(full_o + s, P::TX_BYTES);
      if (NG > 0) tma_load_5d(slot, &tm_gate, x0, y0, z0 + c, 0, (int)bz, full_o + s);
      if (KIND != K_SELF) tma_load_5d(slot + P::OFF_Y, &tm_y, x0, y0, z0 + c, 0, (int)bz, full_o + s);
      if (KIND == K_RK4F) {
        tma_load_5d(slot + P::OFF_A, &tm_A, x0, y0, z0 + c, 0, (int)bz, full_o + s);
        tma_load_5d(slot + P::OFF_B, &tm_B, x0, y0, z0 + c, 0, (int)bz, full_o + s);
      }
    };
    if (producer) {
      while (issued < base_idx + (unsigned)min(nplanes, NSLOT - 1)) { request((int)(issued - base_idx)); ++issued; }
      if (P::ANY)
        while (oissued < obase + (unsigned)min(zlen, NSLOT_O - 1)) { request_op((int)(oissued - obase)); ++oissued; }
    }
    for (int m = 0; m < 2 * R; ++m) arrived(m);

    const int gx = x0 + 2 * lane, gy = y0 + warp;
    const bool live = gx < nx && gy < ny, both = gx + 1 < nx;
    const int hc = (warp + R) * HP + 2 + 2 * lane;   // centre of the pair inside a halo box
    for (int c = 0; c < zlen; ++c) {
      if (producer && issued < base_idx + (unsigned)nplanes && issued < base_idx + (unsigned)(c + NSLOT)) {
        request((int)(issued - base_idx));   // the slot of plane c-1, which every warp released last iteration
        ++issued;
      }
      if (P::ANY && producer && oissued < obase + (unsigned)zlen && oissued < obase + (unsigned)(c + NSLOT_O)) {
        request_op((int)(oissued - obase));
        ++oissued;
      }
      arrived(c + 2 * R);
      const unsigned oidx = obase + (unsigned)c;
      const unsigned char* oslot = r3_smem + P::OFF_OPER + (oidx % (NSLOT_O > 0 ? NSLOT_O : 1)) * P::SLOT_BYTES;
      if (P::ANY) mbar_wait(full_o + oidx % (NSLOT_O > 0 ? NSLOT_O : 1), (oidx / (NSLOT_O > 0 ? NSLOT_O : 1)) & 1u);
      if (rim) {
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // generic writes before the next TMA write
        __syncthreads();   // the patch of the new plane (c = 0: of the first 2r+1 planes) is complete
      }
      if (live) {
        const long long o = mbase + (long long)(z0 + c) * a.g.zstride + (long long)gy * pitch + gx;
        const int pc = warp * TW + 2 * lane;   // the pair inside a tile box
        const double* gs = reinterpret_cast<const double*>(oslot);
        const double* Ys = reinterpret_cast<const double*>(oslot + P::OFF_Y);
        const double* As = reinterpret_cast<const double*>(oslot + P::OFF_A);
        const double* Bs = reinterpret_cast<const double*>(oslot + P::OFF_B);
        double2 zz[NV];
#pragma unroll
        for (int q = ND; q < NV; ++q) zz[q] = ld2(gs + (q - ND) * TSZ + pc);
        const double* hc0 = slot_of(base_idx + (unsigned)(c + R));
        double s0[ND], s1[ND];
#pragma unroll
        for (int q = 0; q < ND; ++q) {
          zz[q] = ld2(hc0 + q * FSZ + hc);
          stencil_pair<STENCIL>(hc0 + q * FSZ, (warp + R) * HP, 2 + 2 * lane, HP, zz[q], s0[q], s1[q]);
          const double2 d1 = ld2(slot_of(base_idx + (unsigned)(c + R - 1)) + q * FSZ + hc);
          const double2 u1 = ld2(slot_of(base_idx + (unsigned)(c + R + 1)) + q * FSZ + hc);
          if (STENCIL == S_LAP9X4) {
            const double2 d2 = ld2(slot_of(base_idx + (unsigned)(c + R - 2)) + q * FSZ + hc);
            const double2 u2 = ld2(slot_of(base_idx + (unsigned)(c + R + 2)) + q * FSZ + hc);
            s0[q] += StencilZ<S_LAP9X4>::apply(zz[q].x, d1.x, u1.x, d2.x, u2.x);
            s1[q] += StencilZ<S_LAP9X4>::apply(zz[q].y, d1.y, u1.y, d2.y, u2.y);
          } else {
            s0[q] += StencilZ<S_LAP5>::apply(zz[q].x, d1.x, u1.x);
            s1[q] += StencilZ<S_LAP5>::apply(zz[q].y, d1.y, u1.y);
          }
        }
        double z0v[NV], z1v[NV], f0[NV], f1[NV];
#pragma unroll
        for (int q = 0; q < NV; ++q) { z0v[q] = zz[q].x; z1v[q] = zz[q].y; }
        MD::reaction(a.p, z0v, f0);
        MD::reaction(a.p, z1v, f1);
#pragma unroll
        for (int q = 0; q < ND; ++q) {
          f0[q] = fma(a.lapw[q], s0[q], f0[q]);
          f1[q] = fma(a.lapw[q], s1[q], f1[q]);
        }
#pragma unroll
        for (int q = 0; q < NV; ++q) {
          double2 yy = make_double2(0.0, 0.0), AA = yy, BB = yy;
          if (KIND != K_SELF) yy = ld2(Ys + q * TSZ + pc);
          if (KIND == K_RK4F) { AA = ld2(As + q * TSZ + pc); BB = ld2(Bs + q * TSZ + pc); }
          const double r0 = combine<KIND>(a.w_y, a.w_in, a.w_A, a.w_B, a.w_f, yy.x, z0v[q], AA.x, BB.x, f0[q]);
          const double r1v = combine<KIND>(a.w_y, a.w_in, a.w_A, a.w_B, a.w_f, yy.y, z1v[q], AA.y, BB.y, f1[q]);
          if (both) st2(a.out + o + q * a.g.fstride, r0, r1v);
          else a.out[o + q * a.g.fstride] = r0;
        }
      }
      // plane c (the lowest of this centre) is not needed any more; at the end of the unit neither are the others
      __syncwarp();
      if (lane == 0) {
        if (P::ANY) mbar_arrive(empty_o + oidx % (NSLOT_O > 0 ? NSLOT_O : 1));
        mbar_arrive(empty + (base_idx + (unsigned)c) % NSLOT);
        if (c == zlen - 1)
          for (int m = zlen; m < nplanes; ++m) mbar_arrive(empty + (base_idx + (unsigned)m) % NSLOT);
      }
    }
    base_idx += (unsigned)nplanes;
    obase += (unsigned)zlen;
  }
}

template <class MD, int STENCIL, int KIND>
cudaError_t run_ring3d(const Problem& pb, const StageLaunch& st, cudaStream_t stream) {
  using L = Oper3D<MD, STENCIL, KIND>;
  using HL = Ring3D<MD, STENCIL>;
  auto kern = ring3d_stage_kernel<MD, STENCIL, KIND>;
  static PerDeviceOnce configured;   // per instantiation and device
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
    if ((e2 = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, NT, L::SMEM_BYTES)) != cudaSuccess) return e2;
    if (occ < 1) return cudaErrorLaunchOutOfResources;
    grid_of[dev].store(sms * occ, std::memory_order_relaxed);
    return cudaSuccess;
  });
  if (e != cudaSuccess) return e;
  Ring3DArgs<MD> ra;
  StageArgs<MD>& a = ra.a;
  a.in = st.in; a.y = st.y ? st.y : st.in; a.A = st.A ? st.A : st.in; a.B = st.B ? st.B : st.in;
  a.out = st.out;
  a.g.nx = pb.nx; a.g.ny = pb.ny; a.g.pitch = pb.pitch; a.g.boundary = pb.boundary;
  a.g.nz = pb.nz; a.g.zstride = pb.zstride;
  a.g.fstride = pb.fstride; a.g.bstride = pb.bstride;
  a.w_y = st.w_y; a.w_in = st.w_in; a.w_A = st.w_A; a.w_B = st.w_B; a.w_f = st.w_f;
  a.dt = pb.dt;
  MD::derive(pb.params, a.p);
  for (int q = 0; q < MD::ND; ++q) a.lapw[q] = a.p.D[q] * stencil_norm(STENCIL) / (pb.dx * pb.dx);
  const long long tiles_x = (pb.nx + TW - 1) / TW, tiles_y = (pb.ny + TH - 1) / TH, chunks = (pb.nz + ZC - 1) / ZC;
  const long long nunits = tiles_x * tiles_y * chunks * pb.batch;
  if (nunits >= (1LL << 31)) return cudaErrorInvalidValue;
  ra.tiles_x = (unsigned)tiles_x;
  ra.nunits = (unsigned)nunits;
  ra.chunks = (int)chunks;
  ra.per_member = make_fastdiv((unsigned)(tiles_x * tiles_y * chunks));
  ra.per_chunk = make_fastdiv((unsigned)(tiles_x * tiles_y));
  ra.per_row = make_fastdiv((unsigned)tiles_x);
  CUtensorMap tm_halo, tm_gate, tm_y, tm_A, tm_B;
  if ((e = tensor_map_5d(a.in, pb, MD::ND, HP, HL::HR, &tm_halo)) != cudaSuccess) return e;
  tm_gate = tm_y = tm_A = tm_B = tm_halo;
  if (L::NG > 0 && (e = tensor_map_5d(a.in + MD::ND * pb.fstride, pb, L::NG, TW, TH, &tm_gate)) != cudaSuccess) return e;
  if (KIND != K_SELF && (e = tensor_map_5d(a.y, pb, MD::NV, TW, TH, &tm_y)) != cudaSuccess) return e;
  if (KIND == K_RK4F) {
    if ((e = tensor_map_5d(a.A, pb, MD::NV, TW, TH, &tm_A)) != cudaSuccess) return e;
    if ((e = tensor_map_5d(a.B, pb, MD::NV, TW, TH, &tm_B)) != cudaSuccess) return e;
  }
  long long grid = grid_of[dev].load(std::memory_order_relaxed);
  if (grid > nunits) grid = nunits;
  kern<<<(unsigned)grid, NT, L::SMEM_BYTES, stream>>>(ra, tm_halo, tm_gate, tm_y, tm_A, tm_B);
  return cudaGetLastError();
}

template <class MD, int STENCIL>
cudaError_t ring3d_by_kind(const Problem& pb, const StageLaunch& st, cudaStream_t s) {
  switch (st.kind) {
    case K_SELF: return run_ring3d<MD, STENCIL, K_SELF>(pb, st, s);
    case K_BASE: return run_ring3d<MD, STENCIL, K_BASE>(pb, st, s);
    case K_RK4F: return run_ring3d<MD, STENCIL, K_RK4F>(pb, st, s);
  }
  return cudaErrorInvalidValue;
}

template <class MD>
cudaError_t ring3d_by_stencil(const Problem& pb, const StageLaunch& st, cudaStream_t s) {
  switch (pb.stencil) {
    case S_LAP5: return ring3d_by_kind<MD, S_LAP5>(pb, st, s);
    case S_LAP9X4: return ring3d_by_kind<MD, S_LAP9X4>(pb, st, s);
  }
  return cudaErrorInvalidValue;
}

}  // namespace

bool stage_ring3d_supported(const Problem& pb, int kind) {
  if (kind != K_SELF && kind != K_BASE && kind != K_RK4F) return false;
  if (pb.nz <= 1 || pb.stencil == S_BOX9) return false;
  const long long nunits = (long long)((pb.nx + TW - 1) / TW) * ((pb.ny + TH - 1) / TH) * ((pb.nz + ZC - 1) / ZC) * pb.batch;
  return nunits < (1LL << 31) && tma_available();
}

cudaError_t launch_stage_ring3d(const Problem& pb, const StageLaunch& st, cudaStream_t stream) {
  if (pb.model == M_FHN) return ring3d_by_stencil<Model<M_FHN, V_PAPER>>(pb, st, stream);
  if (pb.model == M_KARMA)
    return pb.variant == V_TANHFREE ? ring3d_by_stencil<Model<M_KARMA, V_TANHFREE>>(pb, st, stream)
                                    : ring3d_by_stencil<Model<M_KARMA, V_PAPER>>(pb, st, stream);
  if (pb.model == M_BOCF)
    return pb.variant == V_TANHFREE ? ring3d_by_stencil<Model<M_BOCF, V_TANHFREE>>(pb, st, stream)
                                    : ring3d_by_stencil<Model<M_BOCF, V_PAPER>>(pb, st, stream);
  return cudaErrorInvalidValue;
}

}  // namespace cardiac
