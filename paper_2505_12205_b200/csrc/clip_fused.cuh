// clip_fused.cuh -- the whole step as ONE pass over f and g ("D4" of DESIGN.md): k_fused = step_pair of clip_fast.cuh
// plus phi(t+1) = sum_a g+_a(x - e_a, t) (Eq. 38 after streaming, B.4 :990) accumulated ON CHIP from
// the post-collision g+ the block has just computed, so g is never read a second time.
//
// A block owns a TILE: all x of `ty` consecutive lattice rows, planes z0 .. z1-1 (chunk c of the z axis), and walks
// it row by row (one thread = one node pair of the row, as in k_step2).  Source node x' sends g+_a(x') to node
// x' + e_a: 9 target rows (dy, dz); within a target row the three directions (0, +x, -x) are combined by warp
// shuffles, so every thread only ever adds into ITS OWN column pair of a shared-memory ring of 4 planes x (ty+2)
// rows -- no atomics, no per-row barrier (warp edges: lanes 0 / 31 keep private edge accumulators that the
// neighbouring warp's edge lane adds when the plane is flushed).  A ring plane is complete (as far as this tile is
// concerned) once the next plane has been processed; it is then flushed:
//   rows inside the tile            -> phi_dst (own sum; complete for rows not on the tile surface)
//   rows y0-1, y0+ty and the planes z0-1, z1 (the tile's halo) -> `part`, a per-tile partial-sum buffer
// k_fix then adds, in a fixed order, the <= 5 neighbour partials to every row on a tile surface.  Deterministic
// (no floating-point atomics); summation ORDER differs from k_phi2's sum19, so the fields agree with the two-kernel
// path to round-off, not bit for bit (G21).
//
// Walls (halfway bounce-back, B.10-B.11 :1034-1037): a link that would leave through a wall face returns to the
// sending node as the opposite population, i.e. its g+ lands on the sender's own row and column.
#pragma once
#include "clip_fast.cuh"
#include <cooperative_groups.h>

namespace clip {

constexpr int FUSED_SLOTS = 4;  // ring planes of k_fused: z-1, z, z+1 and the one being flushed

constexpr int FUSED_MAX_CHUNKS = 256;

template <typename T> struct FusedP {
  T* phi_dst;             // phi(t+1)                         [nz][ny][nx]
  T* part;                // partial sums of the tile halos   [tiles][2 tzmax + 2 (ty + 2)][nx]
  int ty, ytiles, nchunks, tzmax;
  int zc[FUSED_MAX_CHUNKS + 1];  // chunk c covers the planes zc[c] .. zc[c+1]-1 (sizes <= tzmax; clip.cu: fused_plan)
  long long tile_stride;  // elements of `part` per tile
  int z_wrap;             // the z faces are PERIODIC: the first and the last chunk are neighbours (k_fix)
  int cs;                 // tiles per thread-block cluster along y (k_fused<..., CL = true>; k_fix then skips their shared surfaces); <= 1: none
  int c_mode;             // which chunks a k_fused launch covers: 0 all (c = blockIdx.y), 1 the first and the last one, 2 all others
};
// rows of a tile's slab in `part`
__host__ __device__ __forceinline__ int slot_ym(int k) { return k; }
__host__ __device__ __forceinline__ int slot_yp(int k, int tzmax) { return tzmax + k; }
__host__ __device__ __forceinline__ int slot_zm(int j, int tzmax) { return 2 * tzmax + j; }
__host__ __device__ __forceinline__ int slot_zp(int j, int tzmax, int ty) { return 2 * tzmax + ty + 2 + j; }

template <typename T> __device__ __forceinline__ T shfl_up1(T v) { return __shfl_up_sync(0xffffffffu, v, 1); }
template <typename T> __device__ __forceinline__ T shfl_dn1(T v) { return __shfl_down_sync(0xffffffffu, v, 1); }

// Accumulation of one source row into the ring.  Column-private shared memory: acc[(slot * rows + j) * nx + x0 .. +1].
// The nine contributions are formed in registers first; the shared-memory read-modify-writes are then issued as one
// batch of loads followed by one batch of stores (the rows are distinct, which the compiler cannot know).
// WALLS: 0 = periodic code, 1 = any wall face next to the row, 2 = wall faces in x only, 3 / 4 = the same two on lattices that
// (also) have FREESLIP faces in x / y (as in clip_fast.cuh).  Where a population lands (which direction it then has does not
// matter for phi = sum_a g_a): a link that crosses a WALL face returns to the sender (B.10-B.11); a link that crosses a free-slip
// face keeps its tangential displacement and drops the normal one (B.8-B.9 :1017-1026); a wall crossing anywhere wins.
template <typename T, int WALLS> struct Scatter {
  typedef P2<T> V;
  T* ring;     // ring base
  T* edge_p;   // [slots * rows][nwarps]: lane 31's +x sends (land in the next warp's first column)
  T* edge_m;   // [slots * rows][nwarps]: lane 0's  -x sends (land in the previous warp's last column)
  int nx, rows, nwarps, warp, lane;
  int sm, sc, sp;  // ring slots of the planes z-1, z, z+1
  int j;           // ring row of the source row (ly + 1)
  static constexpr bool YZ = WALLS == 1 || WALLS == 3;   // y / z faces next to the row
  static constexpr bool FS = WALLS >= 3;

  struct Tri { V v0, vp, vm; };  // what one source pair sends to a target row with e_x = 0, +1, -1
  template <int dy, int dz> __device__ __forceinline__ bool behind_wall(const Geo& geo) const {
    // the row (dy, dz) lies behind a wall: everything returns to the sender (B.10-B.11)
    return YZ && ((dy > 0 && geo.byp) || (dy < 0 && geo.bym) || (dz > 0 && geo.bzp) || (dz < 0 && geo.bzm));
  }
  template <int dy> __device__ __forceinline__ bool behind_slip(const Geo& geo) const {
    return WALLS == 3 && ((dy > 0 && geo.syp) || (dy < 0 && geo.sym));
  }
  template <int dy, int dz, int a0, int ap, int am> __device__ __forceinline__ Tri take(const Geo& geo, const V (&g)[Q], V& own) const {
    Tri t; t.v0 = g[a0]; t.vp = g[ap]; t.vm = g[am];
    if (behind_wall<dy, dz>(geo)) { own = own + ((t.v0 + t.vp) + t.vm); t.v0 = V(T(0)); t.vp = V(T(0)); t.vm = V(T(0)); }
    return t;
  }
  // the diagonal rows (dy, dz = +-1) carry one direction each; behind a free-slip y face it lands in the row (0, dz)
  template <int dy, int dz, int a0> __device__ __forceinline__ V take_diag(const Geo& geo, const V (&g)[Q], V& own, Tri& row0dz) const {
    V c = g[a0];
    if (behind_wall<dy, dz>(geo)) { own = own + c; c = V(T(0)); }
    else if (behind_slip<dy>(geo)) { row0dz.v0 = row0dz.v0 + c; c = V(T(0)); }
    return c;
  }
  // x faces, then the three directions of a target row are combined: c = what lands in this thread's columns, ep / em = what
  // lane 31 / lane 0 sends across the warp edge
  __device__ __forceinline__ void finish(const Geo& geo, Tri t, V& own, V& c, T& ep, T& em) const {
    if (WALLS) {  // node x0+1 sending +x through the +x face / node x0 sending -x through the -x face
      if (geo.bxp) { own = own + V(T(0), t.vp.hi()); t.vp = V(t.vp.lo(), T(0)); }
      if (geo.bxm) { own = own + V(t.vm.lo(), T(0)); t.vm = V(T(0), t.vm.hi()); }
      if (FS && geo.sxp) { t.v0 = t.v0 + V(T(0), t.vp.hi()); t.vp = V(t.vp.lo(), T(0)); }
      if (FS && geo.sxm) { t.v0 = t.v0 + V(t.vm.lo(), T(0)); t.vm = V(T(0), t.vm.hi()); }
    }
    T up = shfl_up1(t.vp.hi()), dn = shfl_dn1(t.vm.lo());  // executed by every lane (wall rows are uniform over the block)
    if (lane == 0) up = T(0);
    if (lane == 31) dn = T(0);
    c = (t.v0 + V(up, t.vp.lo())) + V(t.vm.hi(), dn);
    ep = t.vp.hi(); em = t.vm.lo();
  }
  __device__ __forceinline__ void operator()(const Geo& geo, const V (&g)[Q]) const {
    typedef typename PairOf<T>::type U;
    V own(T(0)), c[9];
    T ep[5], em[5];
    Tri yp = take<1, 0, 3, 7, 10>(geo, g, own), ym = take<-1, 0, 4, 9, 8>(geo, g, own);
    Tri zp = take<0, 1, 5, 11, 14>(geo, g, own), zm = take<0, -1, 6, 13, 12>(geo, g, own);
    Tri me = take<0, 0, 0, 1, 2>(geo, g, own);
    c[5] = take_diag<1, 1, 15>(geo, g, own, zp);
    c[6] = take_diag<-1, -1, 16>(geo, g, own, zm);
    c[7] = take_diag<1, -1, 17>(geo, g, own, zm);
    c[8] = take_diag<-1, 1, 18>(geo, g, own, zp);
    if (WALLS == 3) {  // the in-plane rows behind a free-slip y face land in the sender's own row, x displacement kept
      if (geo.syp) { me.v0 = me.v0 + yp.v0; me.vp = me.vp + yp.vp; me.vm = me.vm + yp.vm; yp.v0 = V(T(0)); yp.vp = V(T(0)); yp.vm = V(T(0)); }
      if (geo.sym) { me.v0 = me.v0 + ym.v0; me.vp = me.vp + ym.vp; me.vm = me.vm + ym.vm; ym.v0 = V(T(0)); ym.vp = V(T(0)); ym.vm = V(T(0)); }
    }
    finish(geo, yp, own, c[0], ep[0], em[0]);
    finish(geo, ym, own, c[1], ep[1], em[1]);
    finish(geo, zp, own, c[2], ep[2], em[2]);
    finish(geo, zm, own, c[3], ep[3], em[3]);
    finish(geo, me, own, c[4], ep[4], em[4]);  // own row last: with walls it also collects what bounced back
    c[4] = c[4] + own;
    const int r[9] = {sc * rows + j + 1, sc * rows + j - 1, sp * rows + j, sm * rows + j, sc * rows + j,
                      sp * rows + j + 1, sm * rows + j - 1, sm * rows + j + 1, sp * rows + j - 1};
    U* p[9];
    U o[9];
#pragma unroll
    for (int k = 0; k < 9; ++k) { p[k] = reinterpret_cast<U*>(ring + (size_t)r[k] * nx + geo.x0); o[k] = *p[k]; }
#pragma unroll
    for (int k = 0; k < 9; ++k) *p[k] = (V(o[k]) + c[k]).v;
    if (lane == 0 || lane == 31) {
      T* const e = (lane ? edge_p : edge_m) + warp;
      T t[5];
#pragma unroll
      for (int k = 0; k < 5; ++k) t[k] = e[r[k] * nwarps];
#pragma unroll
      for (int k = 0; k < 5; ++k) e[r[k] * nwarps] = t[k] + (lane ? ep[k] : em[k]);
    }
  }
};

// Flush ring slot `s` (ty + 2 rows): column sums + the neighbouring warps' edge sends; the slot is left zeroed.
// dst_row(j) gives the destination of ring row j (pointer to column 0) or nullptr to drop the row.
template <typename T, typename D>
__device__ __forceinline__ void flush_slot(T* ring, T* edge_p, T* edge_m, int nx, int rows, int nwarps, int warp, int lane,
                                           int x0, int s, D dst_row) {
  typedef P2<T> V;
  typedef typename PairOf<T>::type U;
  const int wl = warp == 0 ? nwarps - 1 : warp - 1, wr = warp == nwarps - 1 ? 0 : warp + 1;
  for (int j = 0; j < rows; ++j) {
    const int row = s * rows + j;
    U* p = reinterpret_cast<U*>(ring + (size_t)row * nx + x0);
    V v = V(*p);
    *p = V(T(0)).v;
    if (lane == 0) { T& e = edge_p[row * nwarps + wl]; v = v + V(e, T(0)); e = T(0); }
    if (lane == 31) { T& e = edge_m[row * nwarps + wr]; v = v + V(T(0), e); e = T(0); }
    T* d = dst_row(j);
    if (d) st_pair<T>(d + x0, v);
  }
}

// Cluster form (k_fused<..., CL = true>): the tiles of a thread-block cluster are neighbours in y.  A halo row that belongs to a tile of
// the same cluster is not written to `part`: the owner of the lattice row adds it -- read from the neighbour's ring through distributed
// shared memory, and zeroed there -- to its own sum before the row goes to phi_dst.  lo_* / hi_*: ring and edge arrays of the lower /
// upper neighbour in the cluster (nullptr: none, that surface goes through `part` as without clusters).
template <typename T, typename D>
__device__ __forceinline__ void flush_slot_cl(T* ring, T* edge_p, T* edge_m, int nx, int rows, int nwarps, int warp, int lane, int x0, int s, D dst_row,
                                              T* lo_ring, T* lo_ep, T* lo_em, T* hi_ring, T* hi_ep, T* hi_em) {
  typedef P2<T> V;
  typedef typename PairOf<T>::type U;
  const int wl = warp == 0 ? nwarps - 1 : warp - 1, wr = warp == nwarps - 1 ? 0 : warp + 1;
  auto take = [&](T* rg, T* ep, T* em, int row) -> V {   // read and zero one row's column pair (+ the warp-edge sends) of a ring
    U* p = reinterpret_cast<U*>(rg + (size_t)row * nx + x0);
    V v = V(*p);
    *p = V(T(0)).v;
    if (lane == 0) { T& e = ep[row * nwarps + wl]; v = v + V(e, T(0)); e = T(0); }
    if (lane == 31) { T& e = em[row * nwarps + wr]; v = v + V(T(0), e); e = T(0); }
    return v;
  };
  for (int j = 0; j < rows; ++j) {
    if ((j == 0 && lo_ring) || (j == rows - 1 && hi_ring)) continue;   // the neighbour takes (and zeroes) this row
    V v = take(ring, edge_p, edge_m, s * rows + j);
    if (j == 1 && lo_ring) v = v + take(lo_ring, lo_ep, lo_em, s * rows + rows - 1);
    if (j == rows - 2 && hi_ring) v = v + take(hi_ring, hi_ep, hi_em, s * rows);
    T* d = dst_row(j);
    if (d) st_pair<T>(d + x0, v);
  }
}

// grid = (ytiles, nchunks); block = nx/2 threads (nx % 64 == 0); dynamic shared memory = ring + edges.
// WALLS (kernel level): 0 = periodic lattice, 1 = lattice with WALL faces, 2 = lattice with FREESLIP (and maybe WALL) faces in x / y
template <typename T, int NX, int WALLS, int MAXT, int MINB, bool CL = false>
__global__ void __launch_bounds__(MAXT, MINB) k_fused(const __grid_constant__ FP<T> FPp, const FusedP<T> U) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const KP<T>& P = FPp.k;
  const int nx = NX ? NX : P.nx;
  const int rows = U.ty + 2;
  const int nwarps = blockDim.x >> 5, warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  T* ring = reinterpret_cast<T*>(smem_raw);
  constexpr int nslots = FUSED_SLOTS;
  T* edge_p = ring + (size_t)nslots * rows * nx;
  T* edge_m = edge_p + nslots * rows * nwarps;
  const int x0 = 2 * threadIdx.x;
  const int iy = blockIdx.x;
  const int c = U.c_mode == 0 ? (int)blockIdx.y : (U.c_mode == 1 ? (blockIdx.y ? U.nchunks - 1 : 0) : (int)blockIdx.y + 1);
  const int y0 = iy * U.ty, z0 = U.zc[c], z1 = U.zc[c + 1];
  const int tz = z1 - z0;
  for (int i = threadIdx.x; i < nslots * rows * (nx + 2 * nwarps); i += blockDim.x) ring[i] = T(0);
  T *lo_ring = nullptr, *lo_ep = nullptr, *lo_em = nullptr, *hi_ring = nullptr, *hi_ep = nullptr, *hi_em = nullptr;
  if constexpr (CL) {   // cluster (cs, 1, 1): rank = blockIdx.x % cs, the tiles iy - 1 / iy + 1 of the same chunk
    namespace cg = cooperative_groups;
    cg::cluster_group cl = cg::this_cluster();
    const unsigned rk = cl.block_rank(), cs = cl.num_blocks();
    if (rk > 0) { lo_ring = cl.map_shared_rank(ring, rk - 1); lo_ep = cl.map_shared_rank(edge_p, rk - 1); lo_em = cl.map_shared_rank(edge_m, rk - 1); }
    if (rk + 1 < cs) { hi_ring = cl.map_shared_rank(ring, rk + 1); hi_ep = cl.map_shared_rank(edge_p, rk + 1); hi_em = cl.map_shared_rank(edge_m, rk + 1); }
    cl.sync();
  } else {
    __syncthreads();
  }
  T* const slab = U.part + (long long)(c * U.ytiles + iy) * U.tile_stride;
  Scatter<T, WALLS == 2 ? 3 : (WALLS ? 1 : 0)> sc;
  sc.ring = ring; sc.edge_p = edge_p; sc.edge_m = edge_m; sc.nx = nx; sc.rows = rows; sc.nwarps = nwarps; sc.warp = warp; sc.lane = lane;
  // flush of plane k (-1 .. tz) of the tile, held in ring slot (k + 1) % slots
  auto flush = [&](int k) {
    const int s = (k + 1) % nslots;
    if (k < 0 || k >= tz) {
      flush_slot<T>(ring, edge_p, edge_m, nx, rows, nwarps, warp, lane, x0, s, [&](int j) -> T* {
        return slab + (long long)(k < 0 ? slot_zm(j, U.tzmax) : slot_zp(j, U.tzmax, U.ty)) * nx;
      });
    } else {
      T* const plane = U.phi_dst + ((long long)(z0 + k) * P.ny + y0) * nx;
      auto dst = [&](int j) -> T* {
        if (j == 0) return slab + (long long)slot_ym(k) * nx;
        if (j == rows - 1) return slab + (long long)slot_yp(k, U.tzmax) * nx;
        return plane + (long long)(j - 1) * nx;
      };
      if constexpr (CL) flush_slot_cl<T>(ring, edge_p, edge_m, nx, rows, nwarps, warp, lane, x0, s, dst, lo_ring, lo_ep, lo_em, hi_ring, hi_ep, hi_em);
      else flush_slot<T>(ring, edge_p, edge_m, nx, rows, nwarps, warp, lane, x0, s, dst);
    }
  };
  // FOUR ring slots for three live planes: the slot flushed after plane lz (plane lz-1) is not touched while plane lz+1
  // is processed, so one barrier per plane suffices (a warp's flush overlaps the other warps' next plane).
#pragma unroll 1
  for (int lz = 0; lz < tz; ++lz) {
    const int z = z0 + lz;
    sc.sm = lz % nslots; sc.sc = (lz + 1) % nslots; sc.sp = (lz + 2) % nslots;
#pragma unroll 1
    for (int ly = 0; ly < U.ty; ++ly) {
      const int y = y0 + ly;
      sc.j = ly + 1;
      int wall_row = 0;  // 1: a y / z wall face next to the row; 2: only the x faces are walls (two tests per link instead of six)
      if constexpr (WALLS) {
        const bool yz = (y == 0 && P.bc[2] != BC_PERIODIC) || (y == P.ny - 1 && P.bc[3] != BC_PERIODIC) ||
                        (z == 0 && P.bc[4] != BC_PERIODIC) || (z == P.nz - 1 && P.bc[5] != BC_PERIODIC);
        wall_row = yz ? 1 : ((P.bc[0] != BC_PERIODIC || P.bc[1] != BC_PERIODIC) ? 2 : 0);
        if (wall_row == 1) {
          step_pair<T, LD_NC, LD_NC, ST_WB, NX, WALLS == 2 ? 3 : 1>(FPp, x0, y, z, NoWait(), sc);
        } else if (wall_row == 2) {
          Scatter<T, WALLS == 2 ? 4 : 2> sx;
          sx.ring = ring; sx.edge_p = edge_p; sx.edge_m = edge_m; sx.nx = nx; sx.rows = rows; sx.nwarps = nwarps; sx.warp = warp; sx.lane = lane;
          sx.sm = sc.sm; sx.sc = sc.sc; sx.sp = sc.sp; sx.j = sc.j;
          step_pair<T, LD_NC, LD_NC, ST_WB, NX, WALLS == 2 ? 4 : 2>(FPp, x0, y, z, NoWait(), sx);
        }
      }
      if (wall_row == 0) {
        Scatter<T, 0> sp;
        sp.ring = ring; sp.edge_p = edge_p; sp.edge_m = edge_m; sp.nx = nx; sp.rows = rows; sp.nwarps = nwarps; sp.warp = warp; sp.lane = lane;
        sp.sm = sc.sm; sp.sc = sc.sc; sp.sp = sc.sp; sp.j = sc.j;
        step_pair<T, LD_NC, LD_NC, ST_WB, NX, 0>(FPp, x0, y, z, NoWait(), sp);
      }
    }
    // also keeps the block's warps on the same plane: without it the kernel is 4 % slower (L1 reuse).  Cluster form: the neighbours'
    // sums of plane lz - 1 are complete, and what they took from this ring during their last flush is zeroed
    if constexpr (CL) cooperative_groups::this_cluster().sync(); else __syncthreads();
    flush(lz - 1);
  }
  flush(tz - 1);
  flush(tz);
  if constexpr (CL) cooperative_groups::this_cluster().sync();   // no block leaves while a neighbour may still read its ring
}

// phi(t+1) of the rows on a tile surface: own sum + the neighbour tiles' partials, fixed order.
// Surface rows of a tile are numbered s = 0 .. 2 tzmax + 2 (ty - 2) - 1: [0, tzmax) the row ly = 0 of plane lz = s;
// [tzmax, 2 tzmax) the row ly = ty-1; then the rows 1 .. ty-2 of the first plane and (if the tile has more than one
// plane) of the last plane.  grid = (ytiles, nchunks, ceil(rows / (FIX_ROWS * rows_per_pass))); block = FIX_THREADS.
constexpr int FIX_ROWS = 4;     // passes per block
constexpr int FIX_THREADS = 128;
// 16-byte accesses: 4 floats / 2 doubles per thread; a block covers rows_per_pass = FIX_THREADS / min(nx / EV, FIX_THREADS)
// surface rows per pass.
template <typename T> struct Vec16;
template <> struct Vec16<float> { typedef float4 type; static constexpr int EV = 4; };
template <> struct Vec16<double> { typedef double2 type; static constexpr int EV = 2; };
__device__ __forceinline__ float4 vadd(float4 a, float4 b) { return make_float4(a.x + b.x, a.y + b.y, a.z + b.z, a.w + b.w); }
__device__ __forceinline__ double2 vadd(double2 a, double2 b) { return make_double2(a.x + b.x, a.y + b.y); }
__host__ __device__ __forceinline__ int fix_threads_per_row(int nx, int ev) { return nx / ev < FIX_THREADS ? nx / ev : FIX_THREADS; }

template <typename T> __global__ void __launch_bounds__(FIX_THREADS) k_fix(const __grid_constant__ FP<T> FPp, const FusedP<T> U) {
  typedef typename Vec16<T>::type W;
  constexpr int EV = Vec16<T>::EV;
  const KP<T>& P = FPp.k;
  const int nx = P.nx;
  const int iy = blockIdx.x, c = blockIdx.y;
  const int z0 = U.zc[c], tz = U.zc[c + 1] - z0;
  const int iym = iy == 0 ? U.ytiles - 1 : iy - 1, iyp = iy == U.ytiles - 1 ? 0 : iy + 1;
  const int cm = c == 0 ? U.nchunks - 1 : c - 1, cp = c == U.nchunks - 1 ? 0 : c + 1;
  auto slab = [&](int cc, int ii, int slot) -> const T* {
    return U.part + (long long)(cc * U.ytiles + ii) * U.tile_stride + (long long)slot * nx;
  };
  const int nrows = 2 * U.tzmax + 2 * (U.ty - 2);
  const int vpr = nx / EV, tv = fix_threads_per_row(nx, EV), rpp = FIX_THREADS / tv;
  const int myrow = threadIdx.x / tv, v0 = threadIdx.x - myrow * tv;
  if (myrow >= rpp) return;
#pragma unroll 1
  for (int i = 0; i < FIX_ROWS; ++i) {
    int s = (blockIdx.z * FIX_ROWS + i) * rpp + myrow, ly, lz;
    if (s >= nrows) return;
    if (s < 2 * U.tzmax) { ly = s < U.tzmax ? 0 : U.ty - 1; lz = s < U.tzmax ? s : s - U.tzmax; if (lz >= tz) continue; }
    else {
      s -= 2 * U.tzmax;
      ly = 1 + (s < U.ty - 2 ? s : s - (U.ty - 2));
      lz = s < U.ty - 2 ? 0 : tz - 1;
      if (s >= U.ty - 2 && tz == 1) continue;
    }
    const int y = iy * U.ty + ly;
    // without z periodicity nothing arrives from beyond the first / the last chunk (walls send nothing there; next to an INLET /
    // OUTLET plane the generic kernels redo the plane, clip.cu)
    const bool ylo = ly == 0, yhi = ly == U.ty - 1;
    const bool zlo = lz == 0 && (U.z_wrap || c > 0), zhi = lz == tz - 1 && (U.z_wrap || c < U.nchunks - 1);
    const T* src[8];
    int ns = 0;
    // (cluster form of k_fused: the surfaces between the tiles of a cluster are already complete)
    if (ylo && (U.cs <= 1 || iy % U.cs == 0)) src[ns++] = slab(c, iym, slot_yp(lz, U.tzmax));
    if (yhi && (U.cs <= 1 || iy % U.cs == U.cs - 1)) src[ns++] = slab(c, iyp, slot_ym(lz));
    if (zlo) src[ns++] = slab(cm, iy, slot_zp(ly + 1, U.tzmax, U.ty));
    if (zhi) src[ns++] = slab(cp, iy, slot_zm(ly + 1, U.tzmax));
    if (ylo && zlo) src[ns++] = slab(cm, iym, slot_zp(U.ty + 1, U.tzmax, U.ty));
    if (ylo && zhi) src[ns++] = slab(cp, iym, slot_zm(U.ty + 1, U.tzmax));
    if (yhi && zlo) src[ns++] = slab(cm, iyp, slot_zp(0, U.tzmax, U.ty));
    if (yhi && zhi) src[ns++] = slab(cp, iyp, slot_zm(0, U.tzmax));
    if (ns == 0) continue;
    T* const row = U.phi_dst + ((long long)(z0 + lz) * P.ny + y) * nx;
    for (int v = v0; v < vpr; v += tv) {
      W a = __ldca(reinterpret_cast<const W*>(row) + v);
      for (int k = 0; k < ns; ++k) a = vadd(a, __ldca(reinterpret_cast<const W*>(src[k]) + v));
      reinterpret_cast<W*>(row)[v] = a;
    }
  }
}

}  // namespace clip
