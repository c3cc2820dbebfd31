// resident.cuh — plan PERSISTENT for grids that fit the shared memory of one thread-block cluster:
// ONE launch advances all nsteps.
//
// The paper's small-grid regime (N < N0 ~ 362, Fig. 5 :166) is bound by the cost of
// launching (n_d + 2) n_s kernels per time step, not by arithmetic.  Here a batch member is owned
// by one cluster of C <= 16 CTAs (8 for batches of more than 4 members) for the whole run; CTA `rank` holds the slab of rows
// [rank h, rank h + h).  The stage values of the diffusing fields live in two shared-memory buffers
// framed by a ghost ring of r cells, each thread owns up to KP fixed x-adjacent pairs of cells and
// keeps their step-start value y, the running RK sum and the gating variables in registers.
// A substep is: stencil + reaction + RK update of the owned cells (buffer `cur` -> `nxt`),
// cluster barrier, refill of the ghost ring of `nxt` — ghost columns from the CTA's own rows, ghost
// rows from the shared memory of the CTA that owns the row the index reflects / wraps / continues
// to, read through distributed shared memory (PAPER.md:104 Fig. 1, :114; Q3) — CTA
// barrier.  Global memory is touched before the first and after the last step only; the
// "lock-step" between substeps is a hardware cluster barrier (~0.2 us) instead of a
// kernel boundary.  Batch members (the nearby trajectories of a Newton-Krylov solve)
// run on different clusters.
//
// The per-cell arithmetic is the instruction sequence of the tile engine (tile.cuh): same
// Stencil<>::apply operand pairing, Model<>::reaction, a_dt / b_dt updates — results are bitwise
// those of plan FUSED.
#pragma once
#include "stage.cuh"
#include "tile.cuh"
#include "tma.cuh"

namespace cardiac {

constexpr int kResidentThreads = 512;
constexpr int kResidentMaxCluster = 16;  // non-portable cluster size (batches of up to 4 members), else 8

template <class MD>
struct ResidentArgs {
  const double* in;
  double* out;
  Geom g;
  long long nsteps;
  int npx;         // pairs per row = ceil(nx / 2)
  int slab;        // rows per CTA = ceil(ny / C)
  int csize;       // C, CTAs per cluster = per batch member
  int sp, sr;      // shared row pitch (doubles, even) and rows per field: 2 npx + 4, slab + 2 r
  double a_dt[4], b_dt[4];
  double lapw[MD::ND];
  typename MD::Params p;
};

CARDIAC_D unsigned cluster_rank() {
  unsigned r;
  asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
  return r;
}
// Full cluster barrier with release / acquire at cluster scope: orders global AND shared memory (ptxas:
// MEMBAR.ALL.GPU before the arrive, CCTL.IVALL after the wait).  Used where global memory is involved
// (after the load, before the exit).
CARDIAC_D void cluster_sync_all() {
  asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
// CPT = cells per thread and unit: 2 = an x-adjacent pair (128-bit shared-memory accesses); 1 = ONE cell, a warp
// holding 32 x-adjacent cells (stencil_cell: the operands of either half of stencil_pair in the same positions, so the
// same bits).  A substep of a small grid is bound by the latency of one warp's dependent instruction sequence, and
// half the sequence in twice the warps halves it.  (Round 2 first split the PAIRS over even and odd warps; the
// row-major cells are 10-15 % faster — FHN Euler 64^2 0.49 -> 0.44 us per step, RK4 2.49 -> 2.10 — with contiguous
// 8-byte accesses instead of every other half of 16-byte ones.)
template <class MD, int STENCIL, int INTEG, int KP, int CPT>
struct ResidentEngine {
  static constexpr int NV = MD::NV, ND = MD::ND, NG = NV - ND;
  static constexpr int R = stencil_radius(STENCIL);
  static constexpr int NS = StepScheme<INTEG, 1>::NS;
  static constexpr bool RK = StepScheme<INTEG, 1>::RK;
  static constexpr int NT = kResidentThreads;
  static constexpr int GX = 2;  // ghost columns kept on each side (>= r; keeps pairs 16-byte aligned)

  static constexpr int GK = 3;  // exchange duties per thread decoded once
  struct Duty;
  struct Patch;

  // The ghost ring of a slab [y0, y0 + rows): ghost columns -r..-1, nx..nx+r-1 of the own rows (source: the own
  // row, reflected / wrapped column) and ghost rows y0-r..y0-1, y0+rows..y0+rows+r-1 over the columns 0..nx-1
  // (source: the CTA that owns the grid row the index reflects / wraps / continues to).  The ring is filled by
  // the OWNER of the source cell (push): a duty = "copy the value at offset `src` of my buffer to offset `dst`
  // of CTA `dest`'s buffer" (dest < 0: my own buffer, a plain shared-memory copy — the ghost columns).
  struct Duty {
    int dst, src, dest;   // dst < 0: none
  };
  struct Patch {
    double y[RK ? KP : 1][CPT][NV];
    double acc[RK ? KP : 1][CPT][NV];
    double g[KP][CPT][NG > 0 ? NG : 1];
    int off[KP];   // offset of the pair inside a shared field, -1 = no such pair (CPT = 1: or no such cell)
    Duty du[GK];   // the first GK duties of this thread
    int more;      // list position from which further duties are decoded on the fly (very wide grids), -1 = none
  };
  // number of CTAs that hold rows
  CARDIAC_D static int active_ctas(const ResidentArgs<MD>& a) { return (a.g.ny + a.slab - 1) / a.slab; }
  // Row duties of CTA `rank`: the ghost ROWS of the CTAs rank-2 .. rank+2 (wrapped on a periodic grid, clipped
  // otherwise; with slabs of at least r rows no other CTA can need a row of this one) whose source row this CTA
  // owns.  At most kMaxRowDuties; written once per launch by one thread into shared memory as triples
  // (destination CTA, offset of the ghost row in its buffer, offset of the source row in mine), field 0, column 0.
  static constexpr int kMaxRowDuties = 5 * 2 * R;
  CARDIAC_D static int build_row_duties(const ResidentArgs<MD>& a, int* tab, int y0, int rank) {
    const int ny = a.g.ny, bc = a.g.boundary, sp = a.sp, ca = active_ctas(a);
    auto target = [&](int oo) -> int {   // the CTA at offset oo - 2, -1 = none
      int D = rank + oo - 2;
      if (bc == B_PERIODIC) { D %= ca; if (D < 0) D += ca; }
      return (D < 0 || D >= ca) ? -1 : D;
    };
    int n = 0;
    for (int o = 0; o < 5; ++o) {
      const int D = target(o);
      bool dup = D < 0;
      for (int oo = 0; oo < o && !dup; ++oo) dup = target(oo) == D;   // the same CTA under a smaller offset
      if (dup) continue;
      const int y0d = D * a.slab, rowsd = min(a.slab, ny - y0d);
      for (int k = 0; k < 2 * R; ++k) {
        const int gy = k < R ? y0d - 1 - k : y0d + rowsd + (k - R);
        const int gs = bidx(gy, ny, bc);          // the grid row it stands for
        if (gs / a.slab != rank) continue;
        tab[3 * n] = D;
        tab[3 * n + 1] = (gy - y0d + R) * sp + GX;
        tab[3 * n + 2] = (gs - y0 + R) * sp + GX;
        ++n;
      }
    }
    return n;
  }
  // Entry e of the duty list: first the ghost columns of the own rows (local copies), then nrd row duties x
  // n_d fields x nx columns.  Every entry is a duty; thread t takes e = t, t + NT, ...
  CARDIAC_D static int duty_count(const ResidentArgs<MD>& a, int rows, int nrd) {
    return rows > 0 ? ND * (2 * R * rows + nrd * a.g.nx) : 0;
  }
  CARDIAC_D static Duty duty_entry(const ResidentArgs<MD>& a, const int* tab, int e, int rows) {
    const int nx = a.g.nx, bc = a.g.boundary, sp = a.sp, fsz = a.sp * a.sr;
    const int ncol = ND * 2 * R * rows;
    Duty d;
    if (e < ncol) {
      const int q = e / (2 * R * rows), f = e - q * (2 * R * rows);
      const int k = f / rows, lr = f - k * rows + R;
      const int gx = k < R ? -1 - k : nx + (k - R);
      d.dst = q * fsz + lr * sp + GX + gx;
      d.src = q * fsz + lr * sp + GX + bidx(gx, nx, bc);
      d.dest = -1;
      return d;
    }
    const int er = e - ncol, i = er / (ND * nx), rem = er - i * (ND * nx), q = rem / nx, gx = rem - q * nx;
    d.dest = tab[3 * i];
    d.dst = q * fsz + tab[3 * i + 1] + gx;
    d.src = q * fsz + tab[3 * i + 2] + gx;
    return d;
  }

  // Complete the ghost ring of buffer `b` in every CTA (exchange number g = 0, 1, ... of this launch).  Call
  // after a CTA barrier (the own interior of `b` is complete); ends with a CTA barrier.
  // Ghost rows travel by st.async: the store lands in the destination CTA's shared memory and completes a
  // transaction count on ITS mbarrier bar[g & 1]; a CTA waits for the 2 r nx n_d values of its own ring and
  // for nobody else — no cluster-wide barrier and no fence between substeps (the async store carries its own
  // release, the wait acquires at cluster scope).  Why two mbarriers: a neighbour that already has all of ITS
  // ghost rows may run one exchange ahead and deliver exchange g+1 while this CTA still waits for another
  // neighbour's exchange g; it cannot be two ahead, because exchange g+2 needs this CTA's rows of g+1.  Why no
  // "buffer free" signal: a CTA pushes after its CTA barrier, i.e. when all of its threads have finished
  // reading the buffer that exchange g+1 of its neighbours will overwrite, and those neighbours need its
  // pushes before they can get there.
  CARDIAC_D static void exchange(const ResidentArgs<MD>& a, double* __restrict__ b, uint64_t* bars, int g, int rows,
                                 int ne, const Patch& st) {
    uint64_t* const bar = bars + (g & 1);
    if (rows > 0 && threadIdx.x == 0) mbar_arrive_expect_tx(bar, (unsigned)(ND * 2 * R * a.g.nx * sizeof(double)));
    auto run_duty = [&](const Duty& d) {
      const double v = b[d.src];
      if (d.dest < 0) {
        b[d.dst] = v;
      } else {
        unsigned raddr, rbar;
        asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(raddr) : "r"(smem_u32(b + d.dst)), "r"(d.dest));
        asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(rbar) : "r"(smem_u32(bar)), "r"(d.dest));
        asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.f64 [%0], %1, [%2];" ::"r"(raddr),
                     "d"(v), "r"(rbar)
                     : "memory");
      }
    };
#pragma unroll
    for (int k = 0; k < GK; ++k)
      if (st.du[k].dst >= 0) run_duty(st.du[k]);
    if (st.more >= 0) {   // very wide grids: more than GK duties per thread, decoded on the fly
      const int* tab = reinterpret_cast<const int*>(bars + 2);
      for (int e = st.more; e < ne; e += NT) run_duty(duty_entry(a, tab, e, rows));
    }
    if (rows > 0) {
      const unsigned parity = (unsigned)(g >> 1) & 1u;
      unsigned ok;
      do {
        asm volatile(
            "{\n\t.reg .pred p;\n\t"
            "mbarrier.try_wait.parity.acquire.cluster.shared::cta.b64 p, [%1], %2;\n\t"
            "selp.u32 %0, 1, 0, p;\n\t}"
            : "=r"(ok)
            : "r"(smem_u32(bar)), "r"(parity)
            : "memory");
      } while (!ok);
    }
    if (STENCIL == S_BOX9) {   // corners: ghost columns of the ghost rows (which have just arrived)
      const int nx = a.g.nx, bc = a.g.boundary, sp = a.sp, fsz = a.sp * a.sr;
      for (int e = threadIdx.x; e < ND * 2 * R * 2 * R && rows > 0; e += NT) {
        const int q = e / (4 * R * R), f = e - q * 4 * R * R, kr = f / (2 * R), kc = f - kr * 2 * R;
        const int lr = kr < R ? R - 1 - kr : R + rows + (kr - R);
        const int gx = kc < R ? -1 - kc : nx + (kc - R);
        double* F = b + q * fsz;
        F[lr * sp + GX + gx] = F[lr * sp + GX + bidx(gx, nx, bc)];
      }
    }
    __syncthreads();
  }

  // unit k of this thread: pair index (CPT = 2) or cell index (CPT = 1) inside the slab, row-major — a warp holds 32
  // x-adjacent units, so its shared-memory accesses are contiguous
  CARDIAC_D static int unit_index(int k) { return threadIdx.x + k * NT; }

  // Substep S of unit k at shared offset o.  W = 2: both cells of the pair (register slots 0, 1);
  // W = 1: the single cell at o (slot 0).
  template <int S, int W>
  CARDIAC_D static void stage_unit(const ResidentArgs<MD>& a, const double* __restrict__ cur,
                                   double* __restrict__ nxt, Patch& st, int k, int o) {
    constexpr bool LAST = (S == NS - 1);
    const int fsz = a.sp * a.sr;
    double2 ctr[ND];
    double s0[ND], s1[ND];
#pragma unroll
    for (int q = 0; q < ND; ++q) {
      if constexpr (W == 2) {
        ctr[q] = ld2(cur + q * fsz + o);
        stencil_pair<STENCIL>(cur + q * fsz, o, 0, a.sp, ctr[q], s0[q], s1[q]);
      } else {
        ctr[q].x = cur[q * fsz + o];
        s0[q] = stencil_cell<STENCIL>(cur + q * fsz, o, a.sp, ctr[q].x);
      }
    }
    double res[2][NV];
#pragma unroll
    for (int h = 0; h < W; ++h) {
      double z[NV], f[NV];
#pragma unroll
      for (int q = 0; q < NV; ++q)
        z[q] = q < ND ? (h == 0 ? ctr[q < ND ? q : 0].x : ctr[q < ND ? q : 0].y)
                      : st.g[k][h][q >= ND ? q - ND : 0];
      MD::reaction(a.p, z, f);
#pragma unroll
      for (int q = 0; q < ND; ++q) f[q] = fma(a.lapw[q], h == 0 ? s0[q] : s1[q], f[q]);
#pragma unroll
      for (int q = 0; q < NV; ++q) {
        double nv;
        if (!RK) {
          nv = fma(a.a_dt[0], f[q], z[q]);
        } else if (LAST) {
          nv = fma(a.b_dt[S], f[q], S == 0 ? st.y[k][h][q] : st.acc[k][h][q]);
          st.y[k][h][q] = nv;   // the next time step starts here
        } else {
          st.acc[k][h][q] = fma(a.b_dt[S], f[q], S == 0 ? st.y[k][h][q] : st.acc[k][h][q]);
          nv = fma(a.a_dt[S], f[q], st.y[k][h][q]);
        }
        res[h][q] = nv;
        if (q >= ND) st.g[k][h][q >= ND ? q - ND : 0] = nv;
      }
    }
#pragma unroll
    for (int q = 0; q < ND; ++q) {
      if (W == 2) st2(nxt + q * fsz + o, res[0][q], res[1][q]);
      else nxt[q * fsz + o] = res[0][q];
    }
  }

  // Substep S of every owned unit: reads `cur`, writes the diffusing fields of `nxt`.
  template <int S>
  CARDIAC_D static void stage(const ResidentArgs<MD>& a, const double* __restrict__ cur,
                              double* __restrict__ nxt, Patch& st) {
    // Units are handed out in order, so the first missing one ends the list.  Leaving the loop there (a branch
    // around the rest) or skipping unit by unit (which lets ptxas predicate and interleave the units of a thread) is
    // the same work; measured, the heavy stages gain from the interleaving (BOCF RK4 96^2 6.2 -> 5.3, 160^2 13.3 ->
    // 12.0, Karma RK4 96^2 as cells 3.8 -> 3.6 us per step) and the light ones lose 3-6 % to it (FHN, Karma as pairs
    // or with Euler).
    constexpr bool kInterleave = NV > 2 || (CPT == 1 && RK);
#pragma unroll
    for (int k = 0; k < KP; ++k) {
      const int o = st.off[k];
      if (o < 0) {
        if (kInterleave) continue;
        break;
      }
      stage_unit<S, CPT>(a, cur, nxt, st, k, o);
    }
  }

  template <int S>
  CARDIAC_D static void stages_from(const ResidentArgs<MD>& a, double* __restrict__ sm, uint64_t* bars, int& cur,
                                    int& g, Patch& st, int rows, int ne) {
    if constexpr (S < NS) {
      const int fsz = a.sp * a.sr;
      double* c = sm + cur * ND * fsz;
      double* n = sm + (cur ^ 1) * ND * fsz;
      stage<S>(a, c, n, st);
      __syncthreads();
      exchange(a, n, bars, g++, rows, ne, st);
      cur ^= 1;
      stages_from<S + 1>(a, sm, bars, cur, g, st, rows, ne);
    }
  }

  // `in` / `out`: the batch member.  Every CTA of the cluster runs this with its own rank.
  CARDIAC_D static void run(const ResidentArgs<MD>& a, const double* __restrict__ in,
                            double* __restrict__ out, double* __restrict__ sm) {
    const int nx = a.g.nx, pitch = a.g.pitch;
    const unsigned rank = cluster_rank();
    const int y0 = (int)rank * a.slab;
    const int rows = max(0, min(a.slab, a.g.ny - y0));
    const int fsz = a.sp * a.sr;
    Patch st;
    // load: diffusing fields -> shared buffer 0, gating fields and y -> registers
    // position of unit k: row of the slab and (first) column; false = no such unit
    auto unit_pos = [&](int k, int& py, int& gx) {
      const int u = unit_index(k), per_row = CPT == 2 ? a.npx : nx;
      if (u >= per_row * rows) return false;
      py = u / per_row;
      gx = CPT * (u - py * per_row);
      return true;
    };
#pragma unroll
    for (int k = 0; k < KP; ++k) {
      int py, gx;
      st.off[k] = -1;
      if (!unit_pos(k, py, gx)) continue;
      st.off[k] = (py + R) * a.sp + GX + gx;
#pragma unroll
      for (int q = 0; q < NV; ++q) {
        const double* f = in + q * a.g.fstride + (long long)(y0 + py) * pitch + gx;
        if constexpr (CPT == 2) {
          double2 v;
          v.x = f[0];
          v.y = gx + 1 < nx ? f[1] : 0.0;
          if (q < ND) st2(sm + q * fsz + st.off[k], v.x, v.y);
          else { st.g[k][0][q >= ND ? q - ND : 0] = v.x; st.g[k][1][q >= ND ? q - ND : 0] = v.y; }
          if (RK) { st.y[k][0][q] = v.x; st.y[k][1][q] = v.y; }
        } else {
          const double v = f[0];
          if (q < ND) sm[q * fsz + st.off[k]] = v;
          else st.g[k][0][q >= ND ? q - ND : 0] = v;
          if (RK) st.y[k][0][q] = v;
        }
      }
    }
    uint64_t* const bars = reinterpret_cast<uint64_t*>(sm + 2 * ND * fsz);
    int* const tab = reinterpret_cast<int*>(bars + 2);   // [0] = number of row duties, then the triples
    if (threadIdx.x == 0) {
      mbar_init(bars, 1);
      mbar_init(bars + 1, 1);
      asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
      tab[3 * kMaxRowDuties] = rows > 0 ? build_row_duties(a, tab, y0, (int)rank) : 0;
    }
    cluster_sync_all();   // the loads are done and every CTA's mbarriers exist before the first push
    const int ne = duty_count(a, rows, tab[3 * kMaxRowDuties]);
    st.more = -1;
#pragma unroll
    for (int k = 0; k < GK; ++k) {   // this thread's exchange duties: the first GK decoded once
      const int e = threadIdx.x + k * NT;
      st.du[k].dst = -1;
      if (e < ne) st.du[k] = duty_entry(a, tab, e, rows);
    }
    if (threadIdx.x + GK * NT < ne) st.more = threadIdx.x + GK * NT;
    int cur = 0, g = 0;
    exchange(a, sm, bars, g++, rows, ne, st);
    for (long long n = 0; n < a.nsteps; ++n) stages_from<0>(a, sm, bars, cur, g, st, rows, ne);
    // store the state: diffusing fields from the current shared buffer, gates from registers
    const double* c = sm + cur * ND * fsz;
#pragma unroll
    for (int k = 0; k < KP; ++k) {
      int py, gx;
      if (!unit_pos(k, py, gx)) continue;
#pragma unroll
      for (int q = 0; q < NV; ++q) {
        double* f = out + q * a.g.fstride + (long long)(y0 + py) * pitch + gx;
        if constexpr (CPT == 2) {
          double2 v;
          if (q < ND) v = ld2(c + q * fsz + st.off[k]);
          else v = make_double2(st.g[k][0][q >= ND ? q - ND : 0], st.g[k][1][q >= ND ? q - ND : 0]);
          f[0] = v.x;
          if (gx + 1 < nx) f[1] = v.y;
        } else {
          f[0] = q < ND ? c[q * fsz + st.off[k]] : st.g[k][0][q >= ND ? q - ND : 0];
        }
      }
    }
    cluster_sync_all();   // nobody leaves while a neighbour may still read its shared memory
  }
};

template <class MD, int STENCIL, int INTEG, int KP, int CPT>
__global__ void __launch_bounds__(kResidentThreads, 1)
    resident_kernel(const __grid_constant__ ResidentArgs<MD> a) {
  extern __shared__ double2 smem_resident[];
  const long long base = (long long)(blockIdx.x / a.csize) * a.g.bstride;
  ResidentEngine<MD, STENCIL, INTEG, KP, CPT>::run(a, a.in + base, a.out + base,
                                              reinterpret_cast<double*>(smem_resident));
}

}  // namespace cardiac
