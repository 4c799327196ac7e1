// clip_fused_tma.cuh -- k_fused with a bulk-async (TMA) feed: the 38 streamed population rows a lattice row needs are copied from
// global to shared memory by `cp.async.bulk` (SASS: UBLKCP), one row ahead of the arithmetic, completion through an mbarrier.
// Bytes in flight then live in shared memory instead of registers (k_fused keeps ~100 loaded values per thread in registers and is
// bound by that, profiles/r02_experiments.md).  Everything else -- tiles, the on-chip phi scatter ring, flushes, k_fix -- is k_fused's.
//
// Layout fact that makes plain (1-D) bulk copies enough: the population buffer is [nz][ny][38][nx], so component c of the lattice row
// (y', z') is ONE contiguous segment of nx words; the x - e_x shift of streaming is applied when the threads read shared memory (the
// whole row is there, periodic wrap included).  Stage layout: [38][nx], slot c = the segment direction c is pulled from, i.e. row
// (y - e_y, z - e_z).  Lattices with all x / y faces PERIODIC only (bounce-back / reflection would need further segments).
#pragma once
#include "clip_fused.cuh"

namespace clip {

__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long* bar, unsigned count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long* bar, unsigned bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, unsigned bytes, unsigned long long* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst)), "l"(src),
               "r"(bytes), "r"(smem_u32(bar))
               : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long* bar, unsigned parity) {
  unsigned ok;
  do {
    asm volatile("{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.u32 %0, 1, 0, p;\n}" : "=r"(ok) : "r"(smem_u32(bar)), "r"(parity) : "memory");
  } while (!ok);
}

constexpr int TMA_STAGES = 2;

// ... or a shared-memory stage that holds the row's 38 source segments (k_fused_tma)
template <typename T> struct StagePull {
  static constexpr bool F_FIRST = false;  // the global loads of u and phi are issued first; then wait for the stage
  const T* stage;  // [38][nx]
  unsigned long long* bar;
  unsigned parity;
  // u and the phi neighbourhood of the row, fetched from global memory while the PREVIOUS row was being computed
  StRaw<T> raw;
  P2<T> u0, u1, u2;
  __device__ __forceinline__ void prefetch(const KP<T>& P, const Geo& geo) {
    u0 = ld_pair<T, LD_NC>(P.u + geo.rc); u1 = ld_pair<T, LD_NC>(P.u + P.n + geo.rc); u2 = ld_pair<T, LD_NC>(P.u + 2 * P.n + geo.rc);
    raw = stencil2_load<T, LD_NC>(P.phi, geo);
  }
  template <typename T2, int HL> __device__ __forceinline__ void load_u(const KP<T2>&, const Geo&, P2<T2>& ux, P2<T2>& uy, P2<T2>& uz) const {
    ux = u0; uy = u1; uz = u2;
  }
  template <typename T2, int HP> __device__ __forceinline__ void stencil(const KP<T2>&, const Geo&, P2<T2>& phi, P2<T2> (&G)[3], P2<T2>& L) const {
    stencil2_eval<T2>(raw, phi, G, L);
  }
  template <typename T2, int HL, int NX, int SET, int WALLS, int a = 0> struct All {
    static __device__ __forceinline__ void run(const T2* __restrict__ st, int nx, const Geo& g, P2<T2> (&v)[Q]) {
      typedef typename PairOf<T2>::type U;
      const T2* __restrict__ r = st + (SET * Q + a) * nx;
      if (cx(a) == 0) v[a] = P2<T2>(*reinterpret_cast<const U*>(r + g.x0));
      else if (cx(a) == 1) v[a] = P2<T2>(r[g.wm ? nx - 1 : g.x0 - 1], r[g.x0]);
      else v[a] = P2<T2>(r[g.x0 + 1], r[g.wp ? 0 : g.x0 + 2]);
      All<T2, HL, NX, SET, WALLS, a + 1>::run(st, nx, g, v);
    }
  };
  template <typename T2, int HL, int NX, int SET, int WALLS> struct All<T2, HL, NX, SET, WALLS, Q> {
    static __device__ __forceinline__ void run(const T2* __restrict__, int, const Geo&, P2<T2> (&)[Q]) {}
  };
  template <typename T2, int HL, int NX, int SET, int WALLS>
  __device__ __forceinline__ void run(const KP<T2>& P, const Geo& geo, P2<T2> (&v)[Q]) const {
    if (SET == 0) mbar_wait(bar, parity);   // the row's segments have landed
    All<T2, HL, NX, SET, WALLS>::run(stage, NX ? NX : P.nx, geo, v);
  }
};

// Hybrid (experiment): f, u and phi from global memory as in k_fused (first load round, in registers), only the 19 g segments -- the
// SECOND load round of step_pair -- through a shared-memory stage [19][nx].
template <typename T> struct StagePullG {
  static constexpr bool F_FIRST = true;
  const T* stage;  // [19][nx]: the g segments
  unsigned long long* bar;
  unsigned parity;
  template <typename T2, int HL, int NX, int SET, int WALLS>
  __device__ __forceinline__ void run(const KP<T2>& P, const Geo& geo, P2<T2> (&v)[Q]) const {
    if (SET == 0) { Pull2All<T2, HL, NX, 0, WALLS>::run(P.p_src, P.nx, geo, v); return; }
    mbar_wait(bar, parity);
    StagePull<T2>::template All<T2, HL, NX, 0, WALLS>::run(stage, NX ? NX : P.nx, geo, v);   // slot a of the g stage
  }
  template <typename T2, int HL> __device__ __forceinline__ void load_u(const KP<T2>& P, const Geo& geo, P2<T2>& ux, P2<T2>& uy, P2<T2>& uz) const {
    GlobalPull().template load_u<T2, HL>(P, geo, ux, uy, uz);
  }
  template <typename T2, int HP> __device__ __forceinline__ void stencil(const KP<T2>& P, const Geo& geo, P2<T2>& phi, P2<T2> (&G)[3], P2<T2>& L) const {
    GlobalPull().template stencil<T2, HP>(P, geo, phi, G, L);
  }
};
template <typename T, int NX, int a = 0> struct IssueRowG {
  static __device__ __forceinline__ void run(const KP<T>& P, const Geo& g0, T* stage, unsigned long long* bar) {
    const int nx = NX ? NX : P.nx;
    const T* src = pop_row<T, -cy(a), -cz(a)>(P.p_src, g0) + (Q + a) * nx;
    bulk_g2s(stage + a * nx, src, (unsigned)(nx * sizeof(T)), bar);
    IssueRowG<T, NX, a + 1>::run(P, g0, stage, bar);
  }
};
template <typename T, int NX> struct IssueRowG<T, NX, Q> {
  static __device__ __forceinline__ void run(const KP<T>&, const Geo&, T*, unsigned long long*) {}
};

// one thread: issue the 38 segment copies of lattice row (y, z) into `stage`
template <typename T, int NX, int c = 0> struct IssueRow {
  static __device__ __forceinline__ void run(const KP<T>& P, const Geo& g0, T* stage, unsigned long long* bar) {
    constexpr int a = c % Q;
    const int nx = NX ? NX : P.nx;
    const T* src = pop_row<T, -cy(a), -cz(a)>(P.p_src, g0) + c * nx;   // g0: geometry of the node pair at x0 = 0
    bulk_g2s(stage + c * nx, src, (unsigned)(nx * sizeof(T)), bar);
    IssueRow<T, NX, c + 1>::run(P, g0, stage, bar);
  }
};
template <typename T, int NX> struct IssueRow<T, NX, NC> {
  static __device__ __forceinline__ void run(const KP<T>&, const Geo&, T*, unsigned long long*) {}
};

// grid = (ytiles, nchunks) as k_fused; dynamic shared memory = ring + edges | stages (128-byte aligned) | mbarriers
// GONLY: the hybrid form (StagePullG): stages of 19 g segments, everything else as k_fused
template <typename T, int NX, int MAXT, int MINB, bool GONLY = false>
__global__ void __launch_bounds__(MAXT, MINB) k_fused_tma(const __grid_constant__ FP<T> FPp, const FusedP<T> U) {
  constexpr int NSEG = GONLY ? Q : NC;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const KP<T>& P = FPp.k;
  const int nx = NX ? NX : P.nx;
  const int rows = U.ty + 2;
  const int nwarps = blockDim.x >> 5, warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  T* ring = reinterpret_cast<T*>(smem_raw);
  constexpr int nslots = FUSED_SLOTS;
  T* edge_p = ring + (size_t)nslots * rows * nx;
  T* edge_m = edge_p + nslots * rows * nwarps;
  const size_t ring_bytes = ((size_t)nslots * rows * (nx + 2 * nwarps) * sizeof(T) + 127) / 128 * 128;
  T* stages = reinterpret_cast<T*>(smem_raw + ring_bytes);
  unsigned long long* full = reinterpret_cast<unsigned long long*>(smem_raw + ring_bytes + (size_t)TMA_STAGES * NSEG * nx * sizeof(T));
  const int x0 = 2 * threadIdx.x;
  const int iy = blockIdx.x;
  const int c = U.c_mode == 0 ? (int)blockIdx.y : (U.c_mode == 1 ? (blockIdx.y ? U.nchunks - 1 : 0) : (int)blockIdx.y + 1);
  const int y0 = iy * U.ty, z0 = U.zc[c], z1 = U.zc[c + 1];
  const int tz = z1 - z0;
  const unsigned row_bytes = (unsigned)(NSEG * nx * sizeof(T));
  if (threadIdx.x == 0) {
    for (int s = 0; s < TMA_STAGES; ++s) mbar_init(full + s, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  for (int i = threadIdx.x; i < nslots * rows * (nx + 2 * nwarps); i += blockDim.x) ring[i] = T(0);
  __syncthreads();
  auto issue = [&](int r) {  // row r of the tile (r = lz * ty + ly) into stage r % TMA_STAGES; thread 0 only
    const int lz = r / U.ty, ly = r - lz * U.ty;
    const Geo g0 = make_geo<T, 0>(P, 0, y0 + ly, z0 + lz);
    unsigned long long* bar = full + (r % TMA_STAGES);
    mbar_expect_tx(bar, row_bytes);
    if (GONLY) IssueRowG<T, NX>::run(P, g0, stages + (size_t)(r % TMA_STAGES) * NSEG * nx, bar);
    else IssueRow<T, NX>::run(P, g0, stages + (size_t)(r % TMA_STAGES) * NSEG * nx, bar);
  };
  const int nrows = tz * U.ty;
  if (threadIdx.x == 0) issue(0);
  T* const slab = U.part + (long long)(c * U.ytiles + iy) * U.tile_stride;
  Scatter<T, 0> sc;
  sc.ring = ring; sc.edge_p = edge_p; sc.edge_m = edge_m; sc.nx = nx; sc.rows = rows; sc.nwarps = nwarps; sc.warp = warp; sc.lane = lane;
  auto flush = [&](int k) {
    const int s = (k + 1) % nslots;
    if (k < 0 || k >= tz) {
      flush_slot<T>(ring, edge_p, edge_m, nx, rows, nwarps, warp, lane, x0, s, [&](int j) -> T* {
        return slab + (long long)(k < 0 ? slot_zm(j, U.tzmax) : slot_zp(j, U.tzmax, U.ty)) * nx;
      });
    } else {
      T* const plane = U.phi_dst + ((long long)(z0 + k) * P.ny + y0) * nx;
      flush_slot<T>(ring, edge_p, edge_m, nx, rows, nwarps, warp, lane, x0, s, [&](int j) -> T* {
        if (j == 0) return slab + (long long)slot_ym(k) * nx;
        if (j == rows - 1) return slab + (long long)slot_yp(k, U.tzmax) * nx;
        return plane + (long long)(j - 1) * nx;
      });
    }
  };
  int r = 0;
  StagePull<T> pl, nxt;
  StagePullG<T> pg;
  if (!GONLY) pl.prefetch(P, make_geo<T, 0>(P, x0, y0, z0));
#pragma unroll 1
  for (int lz = 0; lz < tz; ++lz) {
    const int z = z0 + lz;
    sc.sm = lz % nslots; sc.sc = (lz + 1) % nslots; sc.sp = (lz + 2) % nslots;
#pragma unroll 1
    for (int ly = 0; ly < U.ty; ++ly, ++r) {
      sc.j = ly + 1;
      // the other stage was read for the last time in the previous iteration (barrier below): refill it with the next row
      if (threadIdx.x == 0 && r + 1 < nrows) issue(r + 1);
      T* const st = stages + (size_t)(r % TMA_STAGES) * NSEG * nx;
      if (GONLY) {
        pg.stage = st; pg.bar = full + (r % TMA_STAGES); pg.parity = (unsigned)((r / TMA_STAGES) & 1);
        step_pair<T, LD_NC, LD_NC, ST_WB, NX, 0, NoWait, Scatter<T, 0>, false, StagePullG<T>>(FPp, x0, y0 + ly, z, NoWait(), sc, pg);
      } else {
        pl.stage = st;
        pl.bar = full + (r % TMA_STAGES);
        pl.parity = (unsigned)((r / TMA_STAGES) & 1);
        if (r + 1 < nrows) {  // u and phi of the next row: in flight during this row's arithmetic
          const int ly1 = ly + 1 < U.ty ? ly + 1 : 0, lz1 = ly + 1 < U.ty ? lz : lz + 1;
          nxt.prefetch(P, make_geo<T, 0>(P, x0, y0 + ly1, z0 + lz1));
        }
        step_pair<T, LD_NC, LD_NC, ST_WB, NX, 0, NoWait, Scatter<T, 0>, false, StagePull<T>>(FPp, x0, y0 + ly, z, NoWait(), sc, pl);
        pl.raw = nxt.raw; pl.u0 = nxt.u0; pl.u1 = nxt.u1; pl.u2 = nxt.u2;
      }
      __syncthreads();  // every thread has taken its values out of this stage (and, at a plane's end, finished the plane's scatter)
    }
    flush(lz - 1);
  }
  flush(tz - 1);
  flush(tz);
}

}  // namespace clip
