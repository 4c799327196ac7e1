// clip_tick.cuh -- the step as ONE launch of the two pair-per-thread bodies (phi_pair, step_pair), ordered by tickets so
// that the second read of g+ hits L2 instead of HBM ("D3" of DESIGN.md).
//
// Two jobs per z plane: A(p) = "phi(t+1) of plane p" (pull g+, sum) and B(z) = "macros + collisions of plane z".
// Blocks are enumerated plane by plane ("groups" of tp tiles); B(z) runs a few groups after A(z+1), spinning on
// per-plane completion counters only for blocks with SMALLER indices (handed out earlier, hence resident or done):
// no co-residency assumption.  Between the pull of g+(plane p) by A(p) and its second pull by B(p) lie about two
// planes of traffic (2 x 84 words x nx x ny), far below the 126 MB L2 for the BASELINE lattices.
// Counters are never reset between steps: targets grow with the step number ("epoch"), compared wrap-safe.
#pragma once
#include "clip_fast.cuh"

namespace clip {

struct TickP {
  unsigned* ticket;   // one counter
  unsigned* done_a;   // [nz] finished A blocks per plane, cumulative over steps
  unsigned base;      // ticket value of the first item of this step  = items_per_step * (epoch - 1)
  unsigned target;    // done_a value that marks a finished plane     = tiles_per_plane * epoch
  int tp, gx;         // tiles per plane, tiles per row of tiles
};

__device__ __forceinline__ unsigned ld_volatile_u32(const unsigned* p) {
  unsigned v;
  asm volatile("ld.volatile.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}

// k_tick2: every block does BOTH jobs for one tile: phi(t+1) of plane p = (i + nz - 1) mod nz (if i < nz) and the
// macros + collisions of plane z = i - lag (if i >= lag >= 3), where i = blockIdx.x / tp is the "group" (nz + lag groups).
// B(z) needs the phi planes z-1, z, z+1, which groups <= i - 1 produced: a block only ever waits for blocks with a
// smaller index (handed out earlier, hence resident or finished); a wait longer than ~0.1 s traps instead of hanging.
// All loads of the block (g pull of plane p, f / u of plane z) are in flight before the first use; the second pull
// of g (plane z, read two groups earlier by A) hits L2.  One barrier per block.
template <typename T, int NX, bool WALLS, int MINB>
__global__ void __launch_bounds__(256, MINB) k_tick2(const __grid_constant__ FP<T> FPp, const TickP tk, const int lag) {
  typedef P2<T> V;
  const KP<T>& P = FPp.k;
  const int tid = threadIdx.y * blockDim.x + threadIdx.x;
  const int nz = P.nz;
  const int grp = blockIdx.x / tk.tp, r = blockIdx.x - grp * tk.tp;
  const bool has_a = grp < nz, has_b = grp >= lag;
  const int pa = (grp + nz - 1) % nz, z = grp - lag;
  const int bxi = r % tk.gx, byi = r / tk.gx;
  const int x0 = 2 * (bxi * blockDim.x + threadIdx.x), y = byi * blockDim.y + threadIdx.y;
  unsigned c0 = 0, c1 = 0, c2 = 0;
  const int zm = z <= 0 ? nz - 1 : z - 1, zp = z == nz - 1 ? 0 : z + 1;
  if (has_b && tid == 0) {
    c0 = ld_volatile_u32(tk.done_a + zp); c1 = ld_volatile_u32(tk.done_a + z); c2 = ld_volatile_u32(tk.done_a + zm);
  }
  V ga[Q], f[Q], g[Q], ux, uy, uz;
  Geo geo_a, geo;
  if (has_a) {
    geo_a = make_geo<T, WALLS>(P, x0, y, pa);
    Pull2All<T, LD_NC, NX, 1, WALLS>::run(P.p_src, P.nx, geo_a, ga);
  }
  if (has_b) {
    geo = make_geo<T, WALLS>(P, x0, y, z);
    Pull2All<T, LD_NC, NX, 0, WALLS>::run(P.p_src, P.nx, geo, f);
    ux = ld_pair<T>(P.u + geo.rc); uy = ld_pair<T>(P.u + P.n + geo.rc); uz = ld_pair<T>(P.u + 2 * P.n + geo.rc);
  }
  if (has_a) st_pair<T>(P.phi + geo_a.rc, sum19(ga));
  if (has_b) {
    Pull2All<T, LD_NC, NX, 1, WALLS>::run(P.p_src, P.nx, geo, g);
    if (tid == 0) {
      unsigned spins = 0;
      while ((int)(c0 - tk.target) < 0) { __nanosleep(32); c0 = ld_volatile_u32(tk.done_a + zp); if (++spins > (1u << 21)) __trap(); }
      while ((int)(c1 - tk.target) < 0) { __nanosleep(32); c1 = ld_volatile_u32(tk.done_a + z); if (++spins > (1u << 21)) __trap(); }
      while ((int)(c2 - tk.target) < 0) { __nanosleep(32); c2 = ld_volatile_u32(tk.done_a + zm); if (++spins > (1u << 21)) __trap(); }
      __threadfence();
    }
  }
  __syncthreads();
  if (has_a && tid == 0) { __threadfence(); atomicAdd(tk.done_a + pa, 1u); }
  if (!has_b) return;
  V phi, G[3], L;
  stencil2<T, LD_CA>(P.phi, geo, phi, G, L);
  const Mom2<T> m = moments2<T>(f);
  const Mat2<T> mat = materials2<T>(P, phi, L);
  {  // macros, Alg. 3
    V F[3], D[6];
    total_force2(P, m, mat, ux, uy, uz, G, F, D);
    const V h = V(T(0.5)) * mat.inv_rho;
    ux = fma2(h, F[0], m.mx); uy = fma2(h, F[1], m.my); uz = fma2(h, F[2], m.mz);
  }
  st_pair<T>(P.u + geo.rc, ux); st_pair<T>(P.u + P.n + geo.rc, uy); st_pair<T>(P.u + 2 * P.n + geo.rc, uz);
  collide2<T>(P, m, mat, phi, G, ux, uy, uz, f, g);
  T* const rd = const_cast<T*>(pop_row<T, 0, 0>(P.p_dst, geo));
  Store2All<T, ST_WB, NX, 0>::run(rd, P.nx, f);
  Store2All<T, ST_WB, NX, 1>::run(rd, P.nx, g);
}

}  // namespace clip
