// clip_march.cuh -- the single fused kernel of the fast path ("D2": 2.5-D marching), fully periodic lattices.
//
// A block owns an in-plane tile of TX x TY nodes (TX/2 x TY threads, one node pair per thread) and marches over a
// segment of z planes.  The only non-local dependency of the step, phi(t+1) = sum_a g+_a(x - e_a, t) being needed at
// x and its 18 neighbours before the collision at t+1, is resolved ON CHIP: for plane k+1 the block
// pulls g for its tile AND a one-node halo ring (the ring costs L2 reads, not DRAM: the neighbouring tiles read the
// same lines at about the same time), writes phi(k+1) into a 4-slot shared-memory ring of planes and parks the
// pulled g of its own nodes in a thread-private shared-memory stash; after one barrier, plane k is collided with the
// stencils taken from the ring.  Per lattice update DRAM sees f 19R+19W, g 19R+19W, u 3R+3W, phi 1W = 83 words
// (B_min = 84) instead of 103 for the two-kernel form (k_phi2 + k_step2), plus 2 planes of g per
// z segment.
#pragma once
#include "clip_fast.cuh"

namespace clip {

template <int TX, int TY> struct MarchCfg {
  static constexpr int NT = TX / 2 * TY;                 // threads
  static constexpr int PITCH = TX + 4;                   // phi plane row pitch; interior column lx sits at lx + 2 (even)
  static constexpr int PLANE = PITCH * (TY + 2);         // one phi plane with its halo ring
  static constexpr int RING = 2 * (TX + 2) + 2 * TY;     // halo ring nodes of a tile
  static constexpr int SLOTS = 4;
};

// periodic geometry of a single node (halo ring)
struct Geo1 { int rc, dym, dyp, dzm, dzp, xm, xp; };
template <typename T> __device__ __forceinline__ Geo1 make_geo1(const KP<T>& P, int x, int y, int z) {
  Geo1 g;
  const int nxy = P.nx * P.ny;
  g.rc = (z * P.ny + y) * P.nx + x;
  g.dym = (y == 0) ? (P.ny - 1) * P.nx : -P.nx;
  g.dyp = (y == P.ny - 1) ? -(P.ny - 1) * P.nx : P.nx;
  g.dzm = (z == 0) ? (P.nz - 1) * nxy : -nxy;
  g.dzp = (z == P.nz - 1) ? -(P.nz - 1) * nxy : nxy;
  g.xm = (x == 0) ? P.nx - 1 : -1;
  g.xp = (x == P.nx - 1) ? 1 - P.nx : 1;
  return g;
}
template <typename T, int a> __device__ __forceinline__ T pull1(const T* const (&src)[Q], const Geo1& g) {
  const int i = g.rc + (cy(a) > 0 ? g.dym : (cy(a) < 0 ? g.dyp : 0)) + (cz(a) > 0 ? g.dzm : (cz(a) < 0 ? g.dzp : 0)) +
                (cx(a) > 0 ? g.xm : (cx(a) < 0 ? g.xp : 0));
  return __ldg(src[a] + i);
}
template <typename T, int a = 0> struct Sum1 {
  static __device__ __forceinline__ void run(const T* const (&src)[Q], const Geo1& g, T (&v)[Q]) {
    v[a] = pull1<T, a>(src, g);
    Sum1<T, a + 1>::run(src, g, v);
  }
};
template <typename T> struct Sum1<T, Q> {
  static __device__ __forceinline__ void run(const T* const (&)[Q], const Geo1&, T (&)[Q]) {}
};

// shared-memory pair access
template <typename T> __device__ __forceinline__ P2<T> lds_pair(const T* p);
template <> __device__ __forceinline__ P2<float> lds_pair<float>(const float* p) { return P2<float>(*reinterpret_cast<const float2*>(p)); }
template <> __device__ __forceinline__ P2<double> lds_pair<double>(const double* p) { return P2<double>(*reinterpret_cast<const double2*>(p)); }

template <typename T> __device__ __forceinline__ Row3<T> lds_row3(const T* row) {  // row points at the pair's own column
  Row3<T> r;
  r.C = lds_pair<T>(row);
  r.L = P2<T>(row[-1], r.C.lo());
  r.R = P2<T>(r.C.hi(), row[2]);
  return r;
}

// Eq. 40a/b from the shared-memory planes below / at / above the node pair (same arithmetic as stencil2).
template <typename T, int PITCH>
__device__ __forceinline__ void stencil_smem(const T* pm, const T* pc_, const T* pp, P2<T>& pc, P2<T> (&G)[3], P2<T>& L) {
  typedef P2<T> V;
  const Row3<T> c = lds_row3<T>(pc_), yp = lds_row3<T>(pc_ + PITCH), ym = lds_row3<T>(pc_ - PITCH);
  const Row3<T> zp = lds_row3<T>(pp), zm = lds_row3<T>(pm);
  const V ypzp = lds_pair<T>(pp + PITCH), ymzm = lds_pair<T>(pm - PITCH);
  const V ypzm = lds_pair<T>(pm + PITCH), ymzp = lds_pair<T>(pp - PITCH);
  pc = c.C;
  const V d1 = c.R - pc, d2 = c.L - pc, d3 = yp.C - pc, d4 = ym.C - pc, d5 = zp.C - pc, d6 = zm.C - pc;
  const V d7 = yp.R - pc, d8 = ym.L - pc, d9 = ym.R - pc, d10 = yp.L - pc;
  const V d11 = zp.R - pc, d12 = zm.L - pc, d13 = zm.R - pc, d14 = zp.L - pc;
  const V d15 = ypzp - pc, d16 = ymzm - pc, d17 = ypzm - pc, d18 = ymzp - pc;
  const V s1 = ((d1 + d2) + (d3 + d4)) + (d5 + d6);
  const V s2 = (((d7 + d8) + (d9 + d10)) + ((d11 + d12) + (d13 + d14))) + ((d15 + d16) + (d17 + d18));
  L = fma2(V(T(1.0 / 3.0)), s1, V(T(1.0 / 6.0)) * s2);
  const V e78 = d7 - d8, e910 = d9 - d10, e1112 = d11 - d12, e1314 = d13 - d14, e1516 = d15 - d16, e1718 = d17 - d18;
  G[0] = fma2(V(T(1.0 / 6.0)), d1 - d2, V(T(1.0 / 12.0)) * ((e78 + e910) + (e1112 + e1314)));
  G[1] = fma2(V(T(1.0 / 6.0)), d3 - d4, V(T(1.0 / 12.0)) * ((e78 - e910) + (e1516 + e1718)));
  G[2] = fma2(V(T(1.0 / 6.0)), d5 - d6, V(T(1.0 / 12.0)) * ((e1112 - e1314) + (e1516 - e1718)));
}

template <typename T, int TX, int TY> constexpr size_t march_smem_bytes() {
  typedef MarchCfg<TX, TY> C;
  return (size_t)C::SLOTS * C::PLANE * sizeof(T) + (size_t)2 * Q * C::NT * 2 * sizeof(T);
}

// k_march: grid = (nx/TX, ny/TY, ceil(nz/LZ)); block = TX/2*TY threads; dynamic shared memory = march_smem_bytes.
template <typename T, int TX, int TY, int MINB>
__global__ void __launch_bounds__(MarchCfg<TX, TY>::NT, MINB) k_march(const __grid_constant__ FP<T> FPp, const int LZ) {
  typedef MarchCfg<TX, TY> C;
  typedef P2<T> V;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  T* const ring = reinterpret_cast<T*>(smem_raw);                               // [SLOTS][PLANE]  phi(t+1) planes
  V* const stash = reinterpret_cast<V*>(ring + C::SLOTS * C::PLANE);            // [2][Q][NT]      pulled g of own pair
  const KP<T>& P = FPp.k;
  const int tid = threadIdx.x;
  const int lx0 = 2 * (tid % (TX / 2)), ly = tid / (TX / 2);
  const int x0 = blockIdx.x * TX + lx0, y = blockIdx.y * TY + ly;
  const int z0 = blockIdx.z * LZ;
  const int z1 = min(z0 + LZ, P.nz);
  const int own = (ly + 1) * C::PITCH + lx0 + 2;
  // halo-ring node served by this thread
  const bool has_ring = tid < C::RING;
  int rx = 0, ry = 0, roff = 0;
  if (has_ring) {
    int rlx, rly;
    if (tid < 2 * (TX + 2)) { rly = (tid < TX + 2) ? -1 : TY; rlx = ((tid < TX + 2) ? tid : tid - (TX + 2)) - 1; }
    else { const int j = tid - 2 * (TX + 2); rly = j >> 1; rlx = (j & 1) ? TX : -1; }
    rx = blockIdx.x * TX + rlx; ry = blockIdx.y * TY + rly;
    rx = rx < 0 ? rx + P.nx : (rx >= P.nx ? rx - P.nx : rx);
    ry = ry < 0 ? ry + P.ny : (ry >= P.ny ? ry - P.ny : ry);
    roff = (rly + 1) * C::PITCH + rlx + 2;
  }

  // phase A of plane zp: phi(t+1) of the tile and its ring -> ring slot; pulled g of the own pair -> stash slot
  auto phase_a = [&](int zp, int slot, bool keep, int ss) {
    const Geo ga = make_geo(P, x0, y, zp);
    V g[Q];
    Pull2All<T>::run(FPp.gs, ga, g);
    T gr[Q];
    if (has_ring) {
      const Geo1 g1 = make_geo1(P, rx, ry, zp);
      Sum1<T>::run(FPp.gs, g1, gr);
    }
    T* const pl = ring + slot * C::PLANE;
    *reinterpret_cast<decltype(V().v)*>(pl + own) = sum19(g).v;
    if (has_ring)
      pl[roff] = ((gr[0] + (gr[1] + gr[2])) + ((gr[3] + gr[4]) + (gr[5] + gr[6]))) +
                 (((gr[7] + gr[8]) + (gr[9] + gr[10])) + ((gr[11] + gr[12]) + (gr[13] + gr[14])) + ((gr[15] + gr[16]) + (gr[17] + gr[18])));
    if (keep) {
      V* const st = stash + ss * Q * C::NT + tid;
#pragma unroll
      for (int a = 0; a < Q; ++a) st[a * C::NT] = g[a];
    }
  };

  {
    const int zm = z0 == 0 ? P.nz - 1 : z0 - 1;
    phase_a(zm, (z0 - 1) & 3, false, 0);
    phase_a(z0, z0 & 3, true, z0 & 1);
  }
  for (int k = z0; k < z1; ++k) {
    const Geo geo = make_geo(P, x0, y, k);
    V f[Q];
    Pull2All<T>::run(FPp.fs, geo, f);
    V ux = ld_pair<T>(P.u + geo.rc), uy = ld_pair<T>(P.u + P.n + geo.rc), uz = ld_pair<T>(P.u + 2 * P.n + geo.rc);
    phase_a(k + 1 == P.nz ? 0 : k + 1, (k + 1) & 3, true, (k + 1) & 1);
    __syncthreads();
    // phase B of plane k: macros (Alg. 3) and both collisions (Alg. 1)
    const Mom2<T> m = moments2<T>(f);
    V phi, G[3], L;
    stencil_smem<T, C::PITCH>(ring + ((k - 1) & 3) * C::PLANE + own, ring + (k & 3) * C::PLANE + own,
                              ring + ((k + 1) & 3) * C::PLANE + own, phi, G, L);
    const Mat2<T> mat = materials2<T>(P, phi, L);
    {
      V F[3], D[6];
      total_force2(P, m, mat, ux, uy, uz, G, F, D);
      const V h = V(T(0.5)) * mat.inv_rho;
      ux = fma2(h, F[0], m.mx); uy = fma2(h, F[1], m.my); uz = fma2(h, F[2], m.mz);
    }
    st_pair<T>(P.u + geo.rc, ux); st_pair<T>(P.u + P.n + geo.rc, uy); st_pair<T>(P.u + 2 * P.n + geo.rc, uz);
    st_pair<T>(P.phi + geo.rc, phi);
    V g[Q];
    {
      const V* const st = stash + (k & 1) * Q * C::NT + tid;
#pragma unroll
      for (int a = 0; a < Q; ++a) g[a] = st[a * C::NT];
    }
    collide2<T>(P, m, mat, phi, G, ux, uy, uz, f, g);
    Store2All<T>::run(FPp.fd, geo.rc, f);
    Store2All<T>::run(FPp.gd, geo.rc, g);
  }
}

}  // namespace clip
