// clip_fast.cuh -- fast kernels for lattices with periodic and / or wall faces and even nx: one thread owns the node pair
// (x0, x0+1), all arithmetic two-lane packed (clip_pack.cuh).  Same equations and the same "lean" formulation as
// clip_kernels.cuh (header comment there), reorganised by opposite-direction pairs (a, a+1):
//   f+_a , f+_abar = w_a (A_a +- B_a),  A_a = p* - 1.5 u.u + 4.5 (e_a.u)^2 + k e_a^T D e_a,  B_a = e_a.(3u + 1.5 F/rho)
//   g+_a , g+_abar = (1-w_phi) g + w_a (C_a +- E_a),  C_a = w_phi phi (1 - 1.5 u.u + 4.5 (e_a.u)^2),
//                                                     E_a = e_a.(3 w_phi phi u + (1 - w_phi/2) [1-4(phi-1/2)^2]/W n)
// (Eq. 13, 16-19, 27-28 as read in G2, 33-36).
#pragma once
#include "clip_kernels.cuh"
#include "clip_pack.cuh"

// Compiler-level fence between the two load rounds of step_pair (keeps nvcc from hoisting part of round 2 into round 1
// and splitting round 1 instead; no instruction is emitted).
#ifndef CLIP_LOAD_FENCE
#define CLIP_LOAD_FENCE() asm volatile("" ::: "memory")
#endif

namespace clip {

// Kernel parameters of the fast kernels (kept as a separate type so that their signatures differ from the generic ones).
template <typename T> struct FP { KP<T> k; };

// Per-thread geometry of a node pair on a periodic lattice.  Plain fields (phi, u) are indexed with 32-bit element
// indices (n < 2^31, checked on the host).  The population buffer is [nz][ny][38][nx]: the row of (y', z') starts at
// 38 * (plain row start), so component c of node x0 in the row whose plain index is `row` sits at
// 38 * row - 37 * x0 + c * nx  -- one 64-bit multiply-add per ROW; within a row all 38 components and the x +- 1
// neighbours are constant offsets (load / store immediates when NX is a template parameter).
struct Geo {
  int rc;                  // plain index of node x0 in its own row
  int dym, dyp, dzm, dzp;  // plain offsets to the rows y-1, y+1, z-1, z+1 (periodic wrap, B.5-B.7)
  int xm, xp;              // offsets from x0 to x0-1 and to x0+2 (periodic wrap)
  bool wm, wp;             // x0-1 / x0+2 wrap around
  int x0;
  // walls (WALLS instantiations only): links of this pair that cross a halfway bounce-back face (B.10-B.11) ...
  bool bym, byp, bzm, bzp;  // ... towards y-1, y+1, z-1, z+1 (both nodes of the pair)
  bool bxm, bxp;            // ... towards x0-1 (node x0 only) and towards x0+2 (node x0+1 only)
  // free-slip faces in x / y (WALLS = 3, 4 only; B.8-B.9 :1017-1026): links that are reflected specularly there
  bool sxm, sxp, sym, syp;
  // ... and the phi ghost rule there (clamp = mirror across the wall, R9): plain offsets for the stencil rows / columns
  int cym, cyp, czm, czp, cxm, cxp;
};

// WALLS: 0 = periodic code, 1 = any wall face, 2 = wall faces in x only (blocks away from the y / z faces of a lattice walled in x);
// 3 / 4 = the same two for lattices that (also) have FREESLIP faces in x or y
template <typename T, int WALLS = 0> __device__ __forceinline__ Geo make_geo(const KP<T>& P, int x0, int y, int z) {
  Geo g;
  const int nxy = P.nx * P.ny;
  g.x0 = x0;
  g.rc = (z * P.ny + y) * P.nx + x0;
  g.dym = (y == 0) ? (P.ny - 1) * P.nx : -P.nx;
  g.dyp = (y == P.ny - 1) ? -(P.ny - 1) * P.nx : P.nx;
  g.dzm = (z == 0) ? (P.nz - 1) * nxy : -nxy;
  g.dzp = (z == P.nz - 1) ? -(P.nz - 1) * nxy : nxy;
  g.wm = (x0 == 0); g.wp = (x0 + 2 == P.nx);
  g.xm = g.wm ? P.nx - 1 : -1;
  g.xp = g.wp ? 2 - P.nx : 2;
  g.cym = g.dym; g.cyp = g.dyp; g.czm = g.dzm; g.czp = g.dzp; g.cxm = g.xm; g.cxp = g.xp;
  g.bym = g.byp = g.bzm = g.bzp = g.bxm = g.bxp = false;
  g.sxm = g.sxp = g.sym = g.syp = false;
  if (WALLS == 1 || WALLS == 2) {
    g.bxm = g.wm && P.bc[0] != BC_PERIODIC; g.bxp = g.wp && P.bc[1] != BC_PERIODIC;
    if (WALLS == 1) {
      g.bym = (y == 0) && P.bc[2] != BC_PERIODIC; g.byp = (y == P.ny - 1) && P.bc[3] != BC_PERIODIC;
      g.bzm = (z == 0) && P.bc[4] != BC_PERIODIC; g.bzp = (z == P.nz - 1) && P.bc[5] != BC_PERIODIC;
    }
  }
  if (WALLS >= 3) {
    g.bxm = g.wm && P.bc[0] == BC_WALL; g.bxp = g.wp && P.bc[1] == BC_WALL;
    g.sxm = g.wm && P.bc[0] == BC_FREESLIP; g.sxp = g.wp && P.bc[1] == BC_FREESLIP;
    if (WALLS == 3) {
      g.bym = (y == 0) && P.bc[2] == BC_WALL; g.byp = (y == P.ny - 1) && P.bc[3] == BC_WALL;
      g.sym = (y == 0) && P.bc[2] == BC_FREESLIP; g.syp = (y == P.ny - 1) && P.bc[3] == BC_FREESLIP;
      g.bzm = (z == 0) && P.bc[4] != BC_PERIODIC; g.bzp = (z == P.nz - 1) && P.bc[5] != BC_PERIODIC;
    }
  }
  if (WALLS) {  // phi ghost = mirror value behind walls and free-slip faces alike (R9)
    if (g.bxm || g.sxm) g.cxm = 0;
    if (g.bxp || g.sxp) g.cxp = 1;
    if (g.bym || g.sym) g.cym = 0;
    if (g.byp || g.syp) g.cyp = 0;
    if (g.bzm) g.czm = 0;
    if (g.bzp) g.czp = 0;
  }
  return g;
}
// plain row index of (y + sy, z + sz) under the phi ghost rule
template <int sy, int sz> __device__ __forceinline__ int phi_row_of(const Geo& g) {
  return g.rc + (sy > 0 ? g.cyp : (sy < 0 ? g.cym : 0)) + (sz > 0 ? g.czp : (sz < 0 ? g.czm : 0));
}

// plain row index of (y + sy, z + sz)
template <int sy, int sz> __device__ __forceinline__ int row_of(const Geo& g) {
  return g.rc + (sy > 0 ? g.dyp : (sy < 0 ? g.dym : 0)) + (sz > 0 ? g.dzp : (sz < 0 ? g.dzm : 0));
}
// pointer to component 0 of node x0 in the population row of (y + sy, z + sz)
template <typename T, int sy, int sz> __device__ __forceinline__ const T* pop_row(const T* __restrict__ p, const Geo& g) {
  return p + ((long long)NC * row_of<sy, sz>(g) - (NC - 1) * g.x0);
}

// Streaming (pull, Alg. 2 / B.3-B.6) of direction a of set SET (0: f, 1: g) for the node pair: value at x - e_a.
// NX > 0: nx known at compile time (component offsets become immediates); NX == 0: runtime nx.
// WALLS: a link that crosses a wall face takes the opposite population of the node itself (B.10-B.11; any wall crossing
// wins at edges and corners, R11).
// Every variant is straight-line code: wrap-around and bounce-back SELECT the address of a load, they do not branch around
// it, so that all loads of a node pair can be issued back to back whatever the lattice's faces are.
template <typename T, int a, int H, int NX, int SET, int WALLS>
__device__ __forceinline__ P2<T> pull2(const T* __restrict__ src, int nx_rt, const Geo& g) {
  const int nx = NX ? NX : nx_rt;
  const T* __restrict__ rp = pop_row<T, -cy(a), -cz(a)>(src, g) + (SET * Q + a) * nx;
  if (a == 0) return ld_pair<T, H>(rp);
  const T* __restrict__ own = pop_row<T, 0, 0>(src, g) + (SET * Q + copp(a)) * nx;
  bool rb = false;  // the link crosses a y / z wall: both nodes of the pair take their own opposite population
  if (WALLS == 1 || WALLS == 3) rb = (cy(a) == 1 && g.bym) || (cy(a) == -1 && g.byp) || (cz(a) == 1 && g.bzm) || (cz(a) == -1 && g.bzp);
  // Free-slip (B.8-B.9, pull form, as clip::pull_reflected): a link that crosses a free-slip face was sent with that velocity
  // component reversed by the node that has the SAME coordinate in that dimension; a wall crossing anywhere on the link wins.
  const T* __restrict__ srx = rp;  // source of an x-reflected link: direction (-cx, cy, cz) of the same row
  if (WALLS >= 3) {
    srx = pop_row<T, -cy(a), -cz(a)>(src, g) + (SET * Q + dir_of(-cx(a), cy(a), cz(a))) * nx;
    if (WALLS == 3 && cy(a) != 0) {
      const bool ry = (cy(a) == 1 && g.sym) || (cy(a) == -1 && g.syp);
      const T* __restrict__ r0 = pop_row<T, 0, -cz(a)>(src, g);
      if (ry) { rp = r0 + (SET * Q + dir_of(cx(a), -cy(a), cz(a))) * nx; srx = r0 + (SET * Q + dir_of(-cx(a), -cy(a), cz(a))) * nx; }
    }
  }
  if (cx(a) == 0) return ld_pair<T, H>(rb ? own : rp);
  const T* __restrict__ plo;
  const T* __restrict__ phi;
  if (cx(a) == 1) {
    plo = rp + (g.wm ? nx - 1 : -1); phi = rp;
    if (WALLS >= 3 && g.sxm) plo = srx;
    if (WALLS && g.bxm) plo = own;
  } else {
    plo = rp + 1; phi = rp + (g.wp ? 2 - nx : 2);
    if (WALLS >= 3 && g.sxp) phi = srx + 1;
    if (WALLS && g.bxp) phi = own + 1;
  }
  if (rb) { plo = own; phi = own + 1; }
  return P2<T>(ld_one<T, H>(plo), ld_one<T, H>(phi));
}
template <typename T, int H, int NX, int SET, int WALLS, int a = 0> struct Pull2All {
  static __device__ __forceinline__ void run(const T* __restrict__ src, int nx, const Geo& g, P2<T> (&v)[Q]) {
    v[a] = pull2<T, a, H, NX, SET, WALLS>(src, nx, g);
    Pull2All<T, H, NX, SET, WALLS, a + 1>::run(src, nx, g, v);
  }
};
template <typename T, int H, int NX, int SET, int WALLS> struct Pull2All<T, H, NX, SET, WALLS, Q> {
  static __device__ __forceinline__ void run(const T* __restrict__, int, const Geo&, P2<T> (&)[Q]) {}
};
// stores of set SET into the node pair's own population row `rd` (= pointer to component 0 of node x0)
template <typename T, int H, int NX, int SET, int a = 0> struct Store2All {
  static __device__ __forceinline__ void run(T* __restrict__ rd, int nx_rt, const P2<T> (&v)[Q]) {
    const int nx = NX ? NX : nx_rt;
    st_pair<T, H>(rd + (SET * Q + a) * nx, v[a]);
    Store2All<T, H, NX, SET, a + 1>::run(rd, nx_rt, v);
  }
};
template <typename T, int H, int NX, int SET> struct Store2All<T, H, NX, SET, Q> {
  static __device__ __forceinline__ void run(T* __restrict__, int, const P2<T> (&)[Q]) {}
};

template <typename T> __device__ __forceinline__ P2<T> sum19(const P2<T> (&g)[Q]) {
  return ((g[0] + (g[1] + g[2])) + ((g[3] + g[4]) + (g[5] + g[6]))) +
         (((g[7] + g[8]) + (g[9] + g[10])) + ((g[11] + g[12]) + (g[13] + g[14])) + ((g[15] + g[16]) + (g[17] + g[18])));
}

// phi at x-1, x, x+1 of one row, for both nodes of the pair
template <typename T> struct Row3 { P2<T> L, C, R; };
template <typename T, int H> __device__ __forceinline__ Row3<T> ld_row3(const T* __restrict__ phi, int row, const Geo& g) {
  Row3<T> r;
  r.C = ld_pair<T, H>(phi + row);
  const T m = ld_one<T, H>(phi + (row + g.cxm)), p = ld_one<T, H>(phi + (row + g.cxp));
  r.L = P2<T>(m, r.C.lo());
  r.R = P2<T>(r.C.hi(), p);
  return r;
}

// Eq. 40a/b on differences d = phi(x+e) - phi(x) (exact zero on a uniform field).  Split into the loads
// (StRaw: the 19-point neighbourhood of a node pair) and the arithmetic, so that a kernel may fetch a row ahead (k_fused_tma).
template <typename T> struct StRaw { Row3<T> c, yp, ym, zp, zm; P2<T> ypzp, ymzm, ypzm, ymzp; };
template <typename T, int H = LD_NC> __device__ __forceinline__ StRaw<T> stencil2_load(const T* __restrict__ phi, const Geo& g) {
  StRaw<T> r;
  r.c = ld_row3<T, H>(phi, phi_row_of<0, 0>(g), g);
  r.yp = ld_row3<T, H>(phi, phi_row_of<1, 0>(g), g); r.ym = ld_row3<T, H>(phi, phi_row_of<-1, 0>(g), g);
  r.zp = ld_row3<T, H>(phi, phi_row_of<0, 1>(g), g); r.zm = ld_row3<T, H>(phi, phi_row_of<0, -1>(g), g);
  r.ypzp = ld_pair<T, H>(phi + phi_row_of<1, 1>(g)); r.ymzm = ld_pair<T, H>(phi + phi_row_of<-1, -1>(g));
  r.ypzm = ld_pair<T, H>(phi + phi_row_of<1, -1>(g)); r.ymzp = ld_pair<T, H>(phi + phi_row_of<-1, 1>(g));
  return r;
}
template <typename T> __device__ __forceinline__ void stencil2_eval(const StRaw<T>& r, P2<T>& pc, P2<T> (&G)[3], P2<T>& L) {
  typedef P2<T> V;
  const Row3<T>&c = r.c, &yp = r.yp, &ym = r.ym, &zp = r.zp, &zm = r.zm;
  const V ypzp = r.ypzp, ymzm = r.ymzm, ypzm = r.ypzm, ymzp = r.ymzp;
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
template <typename T, int H = LD_NC>
__device__ __forceinline__ void stencil2(const T* __restrict__ phi, const Geo& g, P2<T>& pc, P2<T> (&G)[3], P2<T>& L) {
  stencil2_eval<T>(stencil2_load<T, H>(phi, g), pc, G, L);
}

template <typename T> struct Mat2 { P2<T> rho, inv_rho, tau, s_nu, mu; };
template <typename T> __device__ __forceinline__ Mat2<T> materials2(const KP<T>& P, P2<T> phi, P2<T> L) {
  typedef P2<T> V;
  Mat2<T> m;
  m.rho = fma2(phi, V(P.drho), V(P.rho_l));                                    // Eq. 39
  m.inv_rho = rcp2(m.rho);
  if (P.visc_interp == 1) m.tau = rcp2(fma2(phi, V(P.itau_h - P.itau_l), V(P.itau_l)));
  else if (P.visc_interp == 2) m.tau = fma2(phi, V(P.rt_h - P.rt_l), V(P.rt_l)) * m.inv_rho;  // Eq. 25: mu linear, tau = 3 mu / rho
  else m.tau = fma2(phi, V(P.tau_h - P.tau_l), V(P.tau_l));                    // Eq. 24
  m.s_nu = rcp2(m.tau + V(T(0.5)));                                            // G3
  m.mu = fms2(V(P.beta4) * phi, (phi - V(T(1))) * (phi - V(T(0.5))), V(P.kappa) * L);  // Eq. 11 (G4)
  return m;
}

template <typename T> struct Mom2 { P2<T> p, mx, my, mz, xx, yy, zz, xy, yz, xz; };
template <typename T> __device__ __forceinline__ Mom2<T> moments2(const P2<T> (&f)[Q]) {
  typedef P2<T> V;
  Mom2<T> m;
  const V s12 = f[1] + f[2], s34 = f[3] + f[4], s56 = f[5] + f[6];
  const V s78 = f[7] + f[8], s910 = f[9] + f[10], s1112 = f[11] + f[12], s1314 = f[13] + f[14];
  const V s1516 = f[15] + f[16], s1718 = f[17] + f[18];
  const V d12 = f[1] - f[2], d34 = f[3] - f[4], d56 = f[5] - f[6];
  const V d78 = f[7] - f[8], d910 = f[9] - f[10], d1112 = f[11] - f[12], d1314 = f[13] - f[14];
  const V d1516 = f[15] - f[16], d1718 = f[17] - f[18];
  const V sxy = s78 + s910, sxz = s1112 + s1314, syz = s1516 + s1718;
  m.p = (f[0] + ((s12 + s34) + s56)) + ((sxy + sxz) + syz);
  m.mx = d12 + ((d78 + d910) + (d1112 + d1314));
  m.my = d34 + ((d78 - d910) + (d1516 + d1718));
  m.mz = d56 + ((d1112 - d1314) + (d1516 - d1718));
  m.xx = s12 + (sxy + sxz);
  m.yy = s34 + (sxy + syz);
  m.zz = s56 + (sxz + syz);
  m.xy = s78 - s910;
  m.xz = s1112 - s1314;
  m.yz = s1516 - s1718;
  return m;
}

// Total force (Eq. 20) and D = dev(Pi^neq); same closed forms as clip::total_force.
// BGK: the trace of Pi^neq relaxes at s_nu too (Eq. 29); WMRT: at rate 1 (Eq. 30)
template <typename T, bool BGK = false>
__device__ __forceinline__ void total_force2(const KP<T>& P, const Mom2<T>& m, const Mat2<T>& mat, P2<T> ux, P2<T> uy,
                                             P2<T> uz, const P2<T> (&G)[3], P2<T> (&F)[3], P2<T> (&D)[6]) {
  typedef P2<T> V;
  const V p3 = m.p * V(T(1.0 / 3.0));
  const V nxx = m.xx - fma2(ux, ux, p3), nyy = m.yy - fma2(uy, uy, p3), nzz = m.zz - fma2(uz, uz, p3);
  const V nxy = m.xy - ux * uy, nyz = m.yz - uy * uz, nxz = m.xz - ux * uz;
  const V tr3 = ((nxx + nyy) + nzz) * V(T(1.0 / 3.0));
  D[0] = nxx - tr3; D[1] = nyy - tr3; D[2] = nzz - tr3; D[3] = nxy; D[4] = nyz; D[5] = nxz;
  const V s = mat.s_nu;
  const V trs = BGK ? s * tr3 : tr3;
  const V Sxx = fma2(s, D[0], trs), Syy = fma2(s, D[1], trs), Szz = fma2(s, D[2], trs);
  const V Sxy = s * D[3], Syz = s * D[4], Sxz = s * D[5];
  const V cmu = -(mat.tau * V(P.drho));
  const V cs = mat.mu - p3 * V(P.drho);
  const V rb = mat.rho - V(P.rho_ref);
  F[0] = fma2(cs, G[0], fma2(rb, V(P.gx), cmu * fma2(Sxx, G[0], fma2(Sxy, G[1], Sxz * G[2]))));
  F[1] = fma2(cs, G[1], fma2(rb, V(P.gy), cmu * fma2(Sxy, G[0], fma2(Syy, G[1], Syz * G[2]))));
  F[2] = fma2(cs, G[2], fma2(rb, V(P.gz), cmu * fma2(Sxz, G[0], fma2(Syz, G[1], Szz * G[2]))));
}

// One opposite pair (a, a+1) of the two collisions.  eu = e_a.u, eDe = e_a^T D e_a, ev = e_a.(3u + h), em = e_a.mvec.
// The f half and the g half are separate so that g can still be in flight while f+ is computed and stored (step_pair).
template <typename T>
struct Coll2 {
  typedef P2<T> V;
  V p, c0, k, omphi, om1;  // p*, -1.5 u.u, 4.5 (1 - s_nu), w_phi phi, 1 - w_phi
  __device__ __forceinline__ V q(V eu) const { return fma2(eu * V(T(4.5)), eu, c0); }  // Gamma_a/w_a - 1 - 3 e.u
  template <int a> __device__ __forceinline__ void pair_f(V eu, V eDe, V ev, V (&f)[Q]) const {
    const V w(cw<T>(a));
    const V A = fma2(k, eDe, p + q(eu));
    f[a] = w * (A + ev);
    f[a + 1] = w * (A - ev);
  }
  // BGK, Eq. 26: f+ = (1 - s) f + s feq_bar + F_a = (1 - s) f + w [s (p* + Gamma'/w) +- e.(3 s u + (2 - s) 1.5 F/rho)];
  // here k = s_nu, c0 = -1.5 u.u, om1 = 1 - s_nu
  template <int a> __device__ __forceinline__ void pair_f_bgk(V eu, V eb, V (&f)[Q]) const {
    const V w(cw<T>(a));
    const V A = k * (p + q(eu));
    f[a] = fma2(om1, f[a], w * (A + eb));
    f[a + 1] = fma2(om1, f[a + 1], w * (A - eb));
  }
  template <int a> __device__ __forceinline__ void pair_g(V eu, V em, V (&g)[Q]) const {
    const V w(cw<T>(a));
    const V C = fma2(omphi, q(eu), omphi);
    g[a] = fma2(om1, g[a], w * (C + em));
    g[a + 1] = fma2(om1, g[a + 1], w * (C - em));
  }
};
// what the g collision needs from the f collision of the same node pair
template <typename T> struct GCtx { Coll2<T> c; P2<T> ux, uy, uz, mx, my, mz, usq15; };

// f collision (Alg. 1) of a node pair: f+ out (a function of the moments only, because the 14 non-shear moments relax at
// rate 1, G2); fills the context of the g collision.
template <typename T, bool BGK = false>
__device__ __forceinline__ void collide2_f(const KP<T>& P, const Mom2<T>& m, const Mat2<T>& mat, P2<T> phi, const P2<T> (&G)[3],
                                           P2<T> ux, P2<T> uy, P2<T> uz, P2<T> (&f)[Q], GCtx<T>& x) {
  typedef P2<T> V;
  V F[3], D[6];
  total_force2<T, BGK>(P, m, mat, ux, uy, uz, G, F, D);
  const V usq15 = V(T(1.5)) * fma2(ux, ux, fma2(uy, uy, uz * uz));
  const V ir15 = V(T(1.5)) * mat.inv_rho;
  // v = 3u + 1.5 F/rho
  const V vx = fma2(V(T(3)), ux, F[0] * ir15), vy = fma2(V(T(3)), uy, F[1] * ir15), vz = fma2(V(T(3)), uz, F[2] * ir15);
  // interface normal (R10) and the F^phi prefactor, Eq. 34
  const V gn = sqrt2(fma2(G[0], G[0], fma2(G[1], G[1], G[2] * G[2]))) + V(T(1e-32));
  const V ph = phi - V(T(0.5));
  const V pref = fma2(V(T(-4)) * ph, ph, V(T(1))) * V(P.inv_W);
  const V cn = (V(T(1) - T(0.5) * P.om_phi) * pref) * rcp2(gn);
  Coll2<T>& c = x.c;
  c.p = m.p; c.c0 = -usq15; c.k = V(T(4.5)) * (V(T(1)) - mat.s_nu);
  c.omphi = V(P.om_phi) * phi; c.om1 = V(T(1) - P.om_phi);
  const V o3 = V(T(3)) * c.omphi;
  x.mx = fma2(o3, ux, cn * G[0]); x.my = fma2(o3, uy, cn * G[1]); x.mz = fma2(o3, uz, cn * G[2]);
  x.ux = ux; x.uy = uy; x.uz = uz; x.usq15 = usq15;
  if (BGK) {  // f is relaxed, not replaced: all 19 pre-collision values are still needed here
    Coll2<T> b;
    b.p = m.p; b.c0 = -usq15; b.k = mat.s_nu; b.om1 = V(T(1)) - mat.s_nu;
    const V s3 = V(T(3)) * mat.s_nu, s2 = V(T(2)) - mat.s_nu;
    const V bx = fma2(s3, ux, s2 * (F[0] * ir15)), by = fma2(s3, uy, s2 * (F[1] * ir15)), bz = fma2(s3, uz, s2 * (F[2] * ir15));
    f[0] = fma2(b.om1, f[0], V(cw<T>(0)) * (mat.s_nu * (m.p - usq15)));
    b.template pair_f_bgk<1>(ux, bx, f);
    b.template pair_f_bgk<3>(uy, by, f);
    b.template pair_f_bgk<5>(uz, bz, f);
    b.template pair_f_bgk<7>(ux + uy, bx + by, f);
    b.template pair_f_bgk<9>(ux - uy, bx - by, f);
    b.template pair_f_bgk<11>(ux + uz, bx + bz, f);
    b.template pair_f_bgk<13>(ux - uz, bx - bz, f);
    b.template pair_f_bgk<15>(uy + uz, by + bz, f);
    b.template pair_f_bgk<17>(uy - uz, by - bz, f);
    return;
  }
  f[0] = V(cw<T>(0)) * (m.p - usq15);
  const V Dxy2 = D[3] + D[3], Dyz2 = D[4] + D[4], Dxz2 = D[5] + D[5];
  const V sxy = D[0] + D[1], sxz = D[0] + D[2], syz = D[1] + D[2];
  c.template pair_f<1>(ux, D[0], vx, f);
  c.template pair_f<3>(uy, D[1], vy, f);
  c.template pair_f<5>(uz, D[2], vz, f);
  c.template pair_f<7>(ux + uy, sxy + Dxy2, vx + vy, f);
  c.template pair_f<9>(ux - uy, sxy - Dxy2, vx - vy, f);
  c.template pair_f<11>(ux + uz, sxz + Dxz2, vx + vz, f);
  c.template pair_f<13>(ux - uz, sxz - Dxz2, vx - vz, f);
  c.template pair_f<15>(uy + uz, syz + Dyz2, vy + vz, f);
  c.template pair_f<17>(uy - uz, syz - Dyz2, vy - vz, f);
}
// g collision (Eq. 33-36): g in/out in place
template <typename T> __device__ __forceinline__ void collide2_g(const GCtx<T>& x, P2<T> (&g)[Q]) {
  typedef P2<T> V;
  const Coll2<T>& c = x.c;
  g[0] = fma2(c.om1, g[0], V(cw<T>(0)) * (c.omphi - c.omphi * x.usq15));
  c.template pair_g<1>(x.ux, x.mx, g);
  c.template pair_g<3>(x.uy, x.my, g);
  c.template pair_g<5>(x.uz, x.mz, g);
  c.template pair_g<7>(x.ux + x.uy, x.mx + x.my, g);
  c.template pair_g<9>(x.ux - x.uy, x.mx - x.my, g);
  c.template pair_g<11>(x.ux + x.uz, x.mx + x.mz, g);
  c.template pair_g<13>(x.ux - x.uz, x.mx - x.mz, g);
  c.template pair_g<15>(x.uy + x.uz, x.my + x.mz, g);
  c.template pair_g<17>(x.uy - x.uz, x.my - x.mz, g);
}

template <typename T>
__device__ __forceinline__ void collide2(const KP<T>& P, const Mom2<T>& m, const Mat2<T>& mat, P2<T> phi, const P2<T> (&G)[3],
                                         P2<T> ux, P2<T> uy, P2<T> uz, P2<T> (&f)[Q], P2<T> (&g)[Q]) {
  GCtx<T> gx;
  collide2_f<T>(P, m, mat, phi, G, ux, uy, uz, f, gx);
  collide2_g<T>(gx, g);
}

// ------------------------------------------------------------------------------------------------ kernels
// Launch shape: blockDim = (bx, by), grid = (ceil(nx/2/bx), ceil(ny/by), nz); thread -> pair (x0, x0+1) of row (y, z).
template <typename T> __device__ __forceinline__ bool pair_coords(const KP<T>& P, int& x0, int& y, int& z) {
  x0 = 2 * (blockIdx.x * blockDim.x + threadIdx.x);
  y = blockIdx.y * blockDim.y + threadIdx.y;
  z = P.z_lo + blockIdx.z;
  return x0 < P.nx && y < P.ny;
}
// Block-uniform: does any node of the block (rows y0 .. y0+rows-1 of plane z, all x) sit next to a wall face?  Blocks
// that do not run the plain periodic code even in a lattice with walls.
template <typename T> __device__ __forceinline__ bool block_touches_wall(const KP<T>& P, int y0, int rows, int z) {
  const int xb = 2 * blockIdx.x * blockDim.x;  // first node column of the block
  return (xb == 0 && P.bc[0] != BC_PERIODIC) || (xb + 2 * (int)blockDim.x >= P.nx && P.bc[1] != BC_PERIODIC) ||
         (y0 == 0 && P.bc[2] != BC_PERIODIC) || (y0 + rows >= P.ny && P.bc[3] != BC_PERIODIC) ||
         (z == 0 && P.bc[4] != BC_PERIODIC) || (z == P.nz - 1 && P.bc[5] != BC_PERIODIC);
}

// Block-uniform: a y or z wall face next to the block (if not, a block of a walled lattice can only meet the x faces: WALLS = 2)
template <typename T> __device__ __forceinline__ bool block_touches_yz_wall(const KP<T>& P, int y0, int rows, int z) {
  return (y0 == 0 && P.bc[2] != BC_PERIODIC) || (y0 + rows >= P.ny && P.bc[3] != BC_PERIODIC) ||
         (z == 0 && P.bc[4] != BC_PERIODIC) || (z == P.nz - 1 && P.bc[5] != BC_PERIODIC);
}

// phi(t+1) = sum_a g_a(x,t+1) (Eq. 38) of one node pair by pulling the post-collision g+(t).
template <typename T, int HG, int NX, int WALLS> __device__ __forceinline__ void phi_pair(const FP<T>& FPp, int x0, int y, int z) {
  const KP<T>& P = FPp.k;
  const Geo geo = make_geo<T, WALLS>(P, x0, y, z);
  P2<T> g[Q];
  Pull2All<T, HG, NX, 1, WALLS>::run(P.p_src, P.nx, geo, g);
  st_pair<T>(P.phi + geo.rc, sum19(g));
}

// One node pair of the step: pull f+, g+ -> macros (Alg. 3) -> both collisions (Alg. 1) -> store f+, g+, u.
// HL: hint of the population / u loads, HP: hint of the phi loads, HS: hint of the stores.  `before_phi()` runs after
// the f loads have been issued and before phi is touched.
// `after(geo, g)` runs last with the post-collision g+ of the pair (the fused kernel accumulates phi(t+1) from it).
// Load schedule (128 registers hold about 75 loaded values, not all 110): round 1 = f, u, phi stencil; the g loads are
// issued as soon as f has been reduced to its 10 moments and phi to (grad, laplacian), and stay in flight while the
// macros and f+ are computed and stored.
struct NoWait { __device__ __forceinline__ void operator()() const {} };
// Where the streamed populations of a node pair come from: global memory (pull2, every kernel but k_fused_tma) ...
struct GlobalPull {
  static constexpr bool F_FIRST = true;   // issue the f loads before u and phi (all of them stay in flight together)
  template <typename T, int HL, int NX, int SET, int WALLS>
  __device__ __forceinline__ void run(const KP<T>& P, const Geo& geo, P2<T> (&v)[Q]) const { Pull2All<T, HL, NX, SET, WALLS>::run(P.p_src, P.nx, geo, v); }
  template <typename T, int HL> __device__ __forceinline__ void load_u(const KP<T>& P, const Geo& geo, P2<T>& ux, P2<T>& uy, P2<T>& uz) const {
    ux = ld_pair<T, HL>(P.u + geo.rc); uy = ld_pair<T, HL>(P.u + P.n + geo.rc); uz = ld_pair<T, HL>(P.u + 2 * P.n + geo.rc);
  }
  template <typename T, int HP> __device__ __forceinline__ void stencil(const KP<T>& P, const Geo& geo, P2<T>& phi, P2<T> (&G)[3], P2<T>& L) const {
    stencil2<T, HP>(P.phi, geo, phi, G, L);
  }
};
struct NoAfter { template <typename T> __device__ __forceinline__ void operator()(const Geo&, const P2<T> (&)[Q]) const {} };
template <typename T, int HL, int HP, int HS, int NX, int WALLS, typename W, typename A = NoAfter, bool BGK = false, typename PL = GlobalPull>
__device__ __forceinline__ void step_pair(const FP<T>& FPp, int x0, int y, int z, W before_phi, A after = A(), PL pl = PL()) {
  typedef P2<T> V;
  const KP<T>& P = FPp.k;
  const Geo geo = make_geo<T, WALLS>(P, x0, y, z);
  V f[Q], g[Q];
  if (PL::F_FIRST) pl.template run<T, HL, NX, 0, WALLS>(P, geo, f);
  V ux, uy, uz;
  pl.template load_u<T, HL>(P, geo, ux, uy, uz);
  before_phi();
  V phi, G[3], L;
  pl.template stencil<T, HP>(P, geo, phi, G, L);
  if (!PL::F_FIRST) pl.template run<T, HL, NX, 0, WALLS>(P, geo, f);   // staged source: u and phi are already on their way
  const Mom2<T> m = moments2<T>(f);
  CLIP_LOAD_FENCE();
  pl.template run<T, HL, NX, 1, WALLS>(P, geo, g);
  const Mat2<T> mat = materials2<T>(P, phi, L);
  {  // macros, Alg. 3: F from (new p*, new phi, lagged u, R13), then Eq. 31b
    V F[3], D[6];
    total_force2<T, BGK>(P, m, mat, ux, uy, uz, G, F, D);
    const V h = V(T(0.5)) * mat.inv_rho;
    ux = fma2(h, F[0], m.mx); uy = fma2(h, F[1], m.my); uz = fma2(h, F[2], m.mz);
  }
  st_pair<T, HS>(P.u + geo.rc, ux); st_pair<T, HS>(P.u + P.n + geo.rc, uy); st_pair<T, HS>(P.u + 2 * P.n + geo.rc, uz);
  GCtx<T> gx;
  collide2_f<T, BGK>(P, m, mat, phi, G, ux, uy, uz, f, gx);
  T* const rd = const_cast<T*>(pop_row<T, 0, 0>(P.p_dst, geo));
  Store2All<T, HS, NX, 0>::run(rd, P.nx, f);
  collide2_g<T>(gx, g);
  Store2All<T, HS, NX, 1>::run(rd, P.nx, g);
  after(geo, g);
}

// WALLS (kernel level): 0 = periodic lattice, 1 = lattice with WALL faces, 2 = lattice with FREESLIP (and maybe WALL) faces in x / y
template <typename T, int NX, int WALLS> __global__ void __launch_bounds__(256) k_phi2(const __grid_constant__ FP<T> FPp) {
  int x0, y, z;
  if (!pair_coords(FPp.k, x0, y, z)) return;
  if (WALLS && !block_touches_wall(FPp.k, y - threadIdx.y, blockDim.y, z)) phi_pair<T, LD_NC, NX, 0>(FPp, x0, y, z);
  else if (WALLS && !block_touches_yz_wall(FPp.k, y - threadIdx.y, blockDim.y, z)) phi_pair<T, LD_NC, NX, WALLS == 2 ? 4 : 2>(FPp, x0, y, z);
  else phi_pair<T, LD_NC, NX, WALLS == 2 ? 3 : (WALLS ? 1 : 0)>(FPp, x0, y, z);
}
// 128-thread blocks; fp32: 3 blocks per SM (<= 168 registers: all ~100 loads of a node pair in flight at once, measured
// faster than 4 blocks at 128 registers), fp64: what 255 registers allow.
// BGK collision (Eq. 26, 29) on the pair kernels: runtime-nx form, periodic / walled lattices (the generic kernels take the rest)
template <typename T, int WALLS, int MINB>
__global__ void __launch_bounds__(128, MINB) k_step2_bgk(const __grid_constant__ FP<T> FPp) {
  int x0, y, z;
  if (!pair_coords(FPp.k, x0, y, z)) return;
  if (WALLS && !block_touches_wall(FPp.k, y - threadIdx.y, blockDim.y, z)) step_pair<T, LD_NC, LD_NC, ST_WB, 0, 0, NoWait, NoAfter, true>(FPp, x0, y, z, NoWait());
  else step_pair<T, LD_NC, LD_NC, ST_WB, 0, WALLS ? 1 : 0, NoWait, NoAfter, true>(FPp, x0, y, z, NoWait());
}
template <typename T, int NX, int WALLS, int MINB>
__global__ void __launch_bounds__(128, MINB) k_step2(const __grid_constant__ FP<T> FPp) {
  int x0, y, z;
  if (!pair_coords(FPp.k, x0, y, z)) return;
  if (WALLS && !block_touches_wall(FPp.k, y - threadIdx.y, blockDim.y, z)) step_pair<T, LD_NC, LD_NC, ST_WB, NX, 0>(FPp, x0, y, z, NoWait());
  else if (WALLS && !block_touches_yz_wall(FPp.k, y - threadIdx.y, blockDim.y, z)) step_pair<T, LD_NC, LD_NC, ST_WB, NX, WALLS == 2 ? 4 : 2>(FPp, x0, y, z, NoWait());
  else step_pair<T, LD_NC, LD_NC, ST_WB, NX, WALLS == 2 ? 3 : (WALLS ? 1 : 0)>(FPp, x0, y, z, NoWait());
}

}  // namespace clip
