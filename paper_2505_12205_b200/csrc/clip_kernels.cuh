// clip_kernels.cuh -- device code of libclip (sm_100a).  See DESIGN.md for the kernel designs and the roofline.
//
// State kept in HBM between steps (SoA, x fastest; T = float or double):
//   pop[cur]        POST-collision populations f+(x,t) (components 0..18) and g+(x,t) (19..37), row-interleaved:
//                   [nz][ny][38][nx] -- the 38 components of one lattice row lie next to each other, so that in the
//                   fast kernels (NX a template parameter) every direction offset is a load/store immediate (A/B buffered)
//   phi             phi(x,t)                                                    [nz][ny][nx]
//   u               u(x,t)                                                   [3][nz][ny][nx]   (node-local update)
//   ob_f, ob_g      PRE-collision populations of the outlet layer z = nz-1 at t   [19][ny][nx] (outlet only)
//   lam             lambda of B.25 for the step in flight (k_outlet_lam)             [ny][nx]  (outlet only)
//   mask            inlet disc mask of the -z face (uint8)                           [ny][nx]  (inlet only)
//
// One step t -> t+1:
//   k_phi : pull g+ (streaming B.4 + all of App. B for g)  ->  phi(t+1) = sum_a g_a   (Eq. 38)
//   k_step: pull f+, g+ (Alg. 2 + App. B) -> macros (Alg. 3) -> both collisions (Alg. 1) -> store f+, g+, u
//
// The arithmetic is the "lean" form of the paper's equations:
//   M^-1 S M = I - (1 - s_nu) P with P_ab = w_a/(2 c_s^4) Q_a : dev(Q_b)   (Eq. 27-28 as read in G2)
//   => f+_a = w_a [p* + 3 e.u + 4.5 (e.u)^2 - 1.5 u.u] + 1.5 w_a (e_a.F)/rho + 4.5 (1 - s_nu) w_a e_a^T D e_a
//      with D = dev(Pi^neq), Pi^neq = sum_a e_a e_a f_a - (p*/3 I + u u)      (Eq. 13, 16, 17, 19)
//   => F_mu = -tau (rho_h - rho_l) [s_nu D + tr(Pi^neq)/3 I] . grad phi          (Eq. 30, 32)
//      g+_a = (1 - w_phi) g_a + w_phi phi Gamma_a + (1 - w_phi/2) F^phi_a        (Eq. 33-36)
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace clip {

enum { BC_PERIODIC = 0, BC_WALL = 1, BC_INLET = 2, BC_OUTLET = 3, BC_FREESLIP = 4 };
constexpr int Q = 19;

// D3Q19 velocity set, Eq. 14; ordering chosen so that the +x set is {1,7,9,11,13}
// and opposite directions are adjacent (a odd -> a+1).
__host__ __device__ constexpr int cx(int a) {
  return (a == 1 || a == 7 || a == 9 || a == 11 || a == 13) ? 1 : ((a == 2 || a == 8 || a == 10 || a == 12 || a == 14) ? -1 : 0);
}
__host__ __device__ constexpr int cy(int a) {
  return (a == 3 || a == 7 || a == 10 || a == 15 || a == 17) ? 1 : ((a == 4 || a == 8 || a == 9 || a == 16 || a == 18) ? -1 : 0);
}
__host__ __device__ constexpr int cz(int a) {
  return (a == 5 || a == 11 || a == 14 || a == 15 || a == 18) ? 1 : ((a == 6 || a == 12 || a == 13 || a == 16 || a == 17) ? -1 : 0);
}
__host__ __device__ constexpr int copp(int a) { return a == 0 ? 0 : ((a & 1) ? a + 1 : a - 1); }
// Eq. 15
template <typename T> __host__ __device__ constexpr T cw(int a) {
  return a == 0 ? T(1.0 / 3.0) : (a < 7 ? T(1.0 / 18.0) : T(1.0 / 36.0));
}

template <typename T> struct KP {
  int nx, ny, nz;
  long long n;    // nodes
  long long nxy;  // nodes per z layer
  int bc[6];
  int has_inlet, has_outlet, any_nonperiodic, visc_interp, collision, phase_only, outlet_u_mode, outlet_clamp, outlet_u_time;
  int z_lo, z_cnt;  // planes [z_lo, z_lo + z_cnt) a k_phi* / k_step* launch covers (whole lattice: 0, nz)
  int z_skip_at, z_skip;  // generic k_phi / k_step: the launch's planes number z_skip_at and up lie z_skip planes further on (the planes next
                          // to an INLET and an OUTLET face in ONE launch); none: z_skip = 0
  T rho_h, rho_l, drho;
  T tau_h, tau_l, itau_h, itau_l, rt_h, rt_l;  // rt = rho tau = 3 mu (Eq. 23, 25)
  T beta4, kappa, inv_W, om_phi;
  T gx, gy, gz, rho_ref;
  T uin[3], phi_in;
  // arrays
  const T* p_src;  // post-collision populations at t     [nz][ny][38][nx]
  T* p_dst;        // post-collision populations at t+1
  T* phi; T* u;
  T* ob_f; T* ob_g; T* lam;
  const uint8_t* mask;
};

template <typename T> __device__ __forceinline__ T rsqrt_(T x);
template <> __device__ __forceinline__ float rsqrt_<float>(float x) { return rsqrtf(x); }
template <> __device__ __forceinline__ double rsqrt_<double>(double x) { return rsqrt(x); }
template <typename T> __device__ __forceinline__ T sqrt_(T x);
template <> __device__ __forceinline__ float sqrt_<float>(float x) { return sqrtf(x); }
template <> __device__ __forceinline__ double sqrt_<double>(double x) { return sqrt(x); }

// ------------------------------------------------------------------------------------------------ geometry
struct Nbr {
  // element offsets to the x-1 / x+1 / y-1 / y+1 / z-1 / z+1 neighbour (periodic wrap applied)
  long long xm, xp, ym, yp, zm, zp;
  // the link towards that side crosses a non-periodic face and bounces back (B.10-B.11)
  bool bxm, bxp, bym, byp, bzm, bzp;
  // the link crosses the inlet disc (unknown, B.4) / the outlet face (layer overwritten, B.5)
  bool ozm, ozp;
  // the link towards that side crosses a free-slip face and is reflected specularly (B.8-B.9)
  bool sxm, sxp, sym, syp, szm, szp;
  bool any;
};

template <typename T>
__device__ __forceinline__ Nbr make_nbr(const KP<T>& P, int x, int y, int z) {
  Nbr b;
  b.xm = (x == 0) ? (long long)(P.nx - 1) : -1LL;
  b.xp = (x == P.nx - 1) ? -(long long)(P.nx - 1) : 1LL;
  b.ym = ((y == 0) ? (long long)(P.ny - 1) : -1LL) * P.nx;
  b.yp = ((y == P.ny - 1) ? -(long long)(P.ny - 1) : 1LL) * P.nx;
  b.zm = ((z == 0) ? (long long)(P.nz - 1) : -1LL) * P.nxy;
  b.zp = ((z == P.nz - 1) ? -(long long)(P.nz - 1) : 1LL) * P.nxy;
  b.bxm = b.bxp = b.bym = b.byp = b.bzm = b.bzp = b.ozm = b.ozp = false;
  b.sxm = b.sxp = b.sym = b.syp = b.szm = b.szp = false;
  if (P.any_nonperiodic) {
    b.bxm = (x == 0) && P.bc[0] == BC_WALL;            b.sxm = (x == 0) && P.bc[0] == BC_FREESLIP;
    b.bxp = (x == P.nx - 1) && P.bc[1] == BC_WALL;     b.sxp = (x == P.nx - 1) && P.bc[1] == BC_FREESLIP;
    b.bym = (y == 0) && P.bc[2] == BC_WALL;            b.sym = (y == 0) && P.bc[2] == BC_FREESLIP;
    b.byp = (y == P.ny - 1) && P.bc[3] == BC_WALL;     b.syp = (y == P.ny - 1) && P.bc[3] == BC_FREESLIP;
    if (z == 0 && P.bc[4] != BC_PERIODIC) {
      const bool disc = (P.bc[4] == BC_INLET) && P.mask[(long long)y * P.nx + x];
      b.szm = P.bc[4] == BC_FREESLIP;
      b.bzm = !disc && !b.szm;
      b.ozm = disc;
    }
    if (z == P.nz - 1 && P.bc[5] != BC_PERIODIC) {
      b.bzp = (P.bc[5] == BC_WALL);
      b.ozp = (P.bc[5] == BC_OUTLET);
      b.szp = (P.bc[5] == BC_FREESLIP);
    }
  }
  b.any = b.bxm | b.bxp | b.bym | b.byp | b.bzm | b.bzp | b.ozm | b.ozp | b.sxm | b.sxp | b.sym | b.syp | b.szm | b.szp;
  return b;
}

constexpr int NC = 2 * Q;  // components per lattice row of the population buffer
// offset, in the population buffer, from a node to the node x - e_a (rows are NC times longer there)
template <int a> __device__ __forceinline__ long long src_off(const Nbr& b) {
  long long o = 0, r = 0;
  if (cx(a) == 1) o += b.xm; else if (cx(a) == -1) o += b.xp;
  if (cy(a) == 1) r += b.ym; else if (cy(a) == -1) r += b.yp;
  if (cz(a) == 1) r += b.zm; else if (cz(a) == -1) r += b.zp;
  return o + NC * r;
}
// index of component 0 of node i (x its column) in the population buffer
__device__ __forceinline__ long long pop_base(long long i, int x) { return (long long)NC * (i - x) + x; }
template <int a> __device__ __forceinline__ bool src_bounce(const Nbr& b) {
  return (cx(a) == 1 && b.bxm) || (cx(a) == -1 && b.bxp) || (cy(a) == 1 && b.bym) || (cy(a) == -1 && b.byp) ||
         (cz(a) == 1 && b.bzm) || (cz(a) == -1 && b.bzp);
}
template <int a> __device__ __forceinline__ bool src_open(const Nbr& b) {
  return (cz(a) == 1 && b.ozm) || (cz(a) == -1 && b.ozp);
}

// Streaming (pull) of one population set at node i: Alg. 2 / B.3-B.4 with periodic wrap (B.5-B.6) and halfway
// bounce-back (B.10-B.11; a wall crossing wins at edges and corners, R11).  Open links (inlet disc / outlet
// face) get 0 and are filled by the caller.
// `src` points at component 0 of the set (f: p_src, g: p_src + Q*nx); pb = pop_base of the node.
// index of the direction with velocity (ex, ey, ez) (must be one of the 19)
__host__ __device__ constexpr int dir_of(int ex, int ey, int ez) {
  for (int a = 0; a < Q; ++a) if (cx(a) == ex && cy(a) == ey && cz(a) == ez) return a;
  return 0;
}
// Free-slip (B.8-B.9), pull form: the population a arriving at a node whose upstream node lies
// behind a free-slip face in dimension d was sent as direction a' = a with component d reversed by the node that has
// the same coordinate in d and the upstream coordinates in the other dimensions (specular reflection half a cell out).
template <typename T, int a, int FX, int FY, int FZ>
__device__ __forceinline__ T pull_reflected(const T* __restrict__ src, int nx, long long pb, const Nbr& b) {
  constexpr int ar = dir_of(FX ? -cx(a) : cx(a), FY ? -cy(a) : cy(a), FZ ? -cz(a) : cz(a));
  long long o = 0, r = 0;
  if (!FX) { if (cx(a) == 1) o += b.xm; else if (cx(a) == -1) o += b.xp; }
  if (!FY) { if (cy(a) == 1) r += b.ym; else if (cy(a) == -1) r += b.yp; }
  if (!FZ) { if (cz(a) == 1) r += b.zm; else if (cz(a) == -1) r += b.zp; }
  return __ldg(src + pb + ar * nx + o + NC * r);
}
template <typename T, int a>
__device__ __forceinline__ T pull_one(const T* __restrict__ src, int nx, long long pb, const Nbr& b, bool slow) {
  if (!slow) return __ldg(src + pb + a * nx + src_off<a>(b));
  if (src_bounce<a>(b)) return __ldg(src + pb + copp(a) * nx);  // a no-slip crossing wins at edges and corners (R11)
  if (src_open<a>(b)) return T(0);
  const bool fx = (cx(a) == 1 && b.sxm) || (cx(a) == -1 && b.sxp);
  const bool fy = (cy(a) == 1 && b.sym) || (cy(a) == -1 && b.syp);
  const bool fz = (cz(a) == 1 && b.szm) || (cz(a) == -1 && b.szp);
  if (fx | fy | fz) {  // D3Q19: at most two components are non-zero
    if (fx && fy) return pull_reflected<T, a, 1, 1, 0>(src, nx, pb, b);
    if (fx && fz) return pull_reflected<T, a, 1, 0, 1>(src, nx, pb, b);
    if (fy && fz) return pull_reflected<T, a, 0, 1, 1>(src, nx, pb, b);
    if (fx) return pull_reflected<T, a, 1, 0, 0>(src, nx, pb, b);
    if (fy) return pull_reflected<T, a, 0, 1, 0>(src, nx, pb, b);
    return pull_reflected<T, a, 0, 0, 1>(src, nx, pb, b);
  }
  return __ldg(src + pb + a * nx + src_off<a>(b));
}

template <typename T, int a = 0> struct PullAll {
  static __device__ __forceinline__ void run(const T* __restrict__ src, int nx, long long pb, const Nbr& b, bool slow,
                                              T (&v)[Q]) {
    v[a] = pull_one<T, a>(src, nx, pb, b, slow);
    PullAll<T, a + 1>::run(src, nx, pb, b, slow, v);
  }
};
template <typename T> struct PullAll<T, Q> {
  static __device__ __forceinline__ void run(const T* __restrict__, int, long long, const Nbr&, bool, T (&)[Q]) {}
};

// Gamma_a / w_a, Eq. 18
template <typename T, int a> __device__ __forceinline__ T gamma_over_w(T ux, T uy, T uz, T usq15) {
  const T eu = T(cx(a)) * ux + T(cy(a)) * uy + T(cz(a)) * uz;
  return T(1) + T(3) * eu + T(4.5) * eu * eu - usq15;
}

// Velocity inlet for g on a disc node (B.16-B.20 as read in G6): unknown set e_z = +1.
template <typename T> __device__ __forceinline__ void inlet_g(const KP<T>& P, T (&g)[Q]) {
  const T ux = P.uin[0], uy = P.uin[1], uz = P.uin[2];
  const T usq15 = T(1.5) * (ux * ux + uy * uy + uz * uz);
  T geq[Q];
#pragma unroll
  for (int a = 0; a < Q; ++a) {
    const T eu = T(cx(a)) * ux + T(cy(a)) * uy + T(cz(a)) * uz;
    geq[a] = P.phi_in * cw<T>(a) * (T(1) + T(3) * eu + T(4.5) * eu * eu - usq15);
  }
  T theta = 0;
#pragma unroll
  for (int a = 0; a < Q; ++a) if (cz(a) == 0) theta += g[a] - geq[a];
#pragma unroll
  for (int a = 0; a < Q; ++a) if (cz(a) == 1) {
    const int b = copp(a);
    g[a] = geq[a] - (g[b] - geq[b]) - ((cx(a) != 0 || cy(a) != 0) ? theta * T(0.25) : T(0));
  }
}
// Velocity inlet for f (B.12-B.15 as read in G6; F = 0 at the inlet so f' = f).
template <typename T> __device__ __forceinline__ void inlet_f(const KP<T>& P, T (&f)[Q]) {
  const T ux = P.uin[0], uy = P.uin[1], uz = P.uin[2];
  T Mx = 0, My = 0;
#pragma unroll
  for (int a = 0; a < Q; ++a) if (cz(a) == 0) { Mx += T(cx(a)) * f[a]; My += T(cy(a)) * f[a]; }
  Mx -= T(2.0 / 3.0) * ux; My -= T(2.0 / 3.0) * uy;
#pragma unroll
  for (int a = 0; a < Q; ++a) if (cz(a) == 1) {
    const T eu = T(cx(a)) * ux + T(cy(a)) * uy + T(cz(a)) * uz;
    f[a] = f[copp(a)] + T(6) * cw<T>(a) * eu - T(0.5) * (T(cx(a)) * Mx + T(cy(a)) * My);
  }
}

// Post-stream, post-BC populations of node (x,y,z) at t+1 (steps 7-9 of DESIGN.md): pull, inlet, outlet.  The outlet's lambda
// is read from P.lam (k_outlet_lam, launched before the kernels of a step).  OUTLET_RULE = false: the post-stream values of
// the node itself even on the outlet layer (k_outlet_lam pulls layer N-1 this way).
template <typename T, bool WITH_F, bool OUTLET_RULE = true>
__device__ __forceinline__ void load_node(const KP<T>& P, int x, int y, int z, T (&f)[Q], T (&g)[Q]) {
  const bool outlet_layer = OUTLET_RULE && P.has_outlet && (z == P.nz - 1);
  const int zs = outlet_layer ? z - 1 : z;  // B.26-B.27 need the post-stream values of layer N-1
  const long long i = (long long)zs * P.nxy + (long long)y * P.nx + x;
  const Nbr b = make_nbr(P, x, y, zs);
  const bool slow = P.any_nonperiodic && b.any;
  const long long pb = pop_base(i, x);
  PullAll<T>::run(P.p_src + Q * P.nx, P.nx, pb, b, slow, g);
  if (WITH_F) PullAll<T>::run(P.p_src, P.nx, pb, b, slow, f);
  if (P.has_inlet && b.ozm) {
    inlet_g(P, g);
    if (WITH_F) inlet_f(P, f);
  }
  if (outlet_layer) {
    const long long c = (long long)y * P.nx + x;
    const T lam = P.lam[c];
    const T inv = T(1) / (T(1) + lam);
#pragma unroll
    for (int a = 0; a < Q; ++a) {
      g[a] = (P.ob_g[a * P.nxy + c] + lam * g[a]) * inv;
      if (WITH_F) f[a] = (P.ob_f[a * P.nxy + c] + lam * f[a]) * inv;
    }
  }
}

// ------------------------------------------------------------------------------------------------ stencils
// Eq. 40a/b on differences d_a = phi(x+e_a) - phi(x); ghost rule: periodic wrap (B.7) or
// clamp at non-periodic faces (R9).
template <typename T>
__device__ __forceinline__ void phi_stencil(const KP<T>& P, const T* __restrict__ phi, int x, int y, int z, T pc,
                                            T (&G)[3], T& L) {
  const long long i = (long long)z * P.nxy + (long long)y * P.nx + x;
  long long oxm = (x == 0) ? ((P.bc[0] == BC_PERIODIC) ? (long long)(P.nx - 1) : 0LL) : -1LL;
  long long oxp = (x == P.nx - 1) ? ((P.bc[1] == BC_PERIODIC) ? -(long long)(P.nx - 1) : 0LL) : 1LL;
  long long oym = ((y == 0) ? ((P.bc[2] == BC_PERIODIC) ? (long long)(P.ny - 1) : 0LL) : -1LL) * P.nx;
  long long oyp = ((y == P.ny - 1) ? ((P.bc[3] == BC_PERIODIC) ? -(long long)(P.ny - 1) : 0LL) : 1LL) * P.nx;
  long long ozm = ((z == 0) ? ((P.bc[4] == BC_PERIODIC) ? (long long)(P.nz - 1) : 0LL) : -1LL) * P.nxy;
  long long ozp = ((z == P.nz - 1) ? ((P.bc[5] == BC_PERIODIC) ? -(long long)(P.nz - 1) : 0LL) : 1LL) * P.nxy;
  T d[Q];
#pragma unroll
  for (int a = 1; a < Q; ++a) {
    long long o = 0;
    if (cx(a) == 1) o += oxp; else if (cx(a) == -1) o += oxm;
    if (cy(a) == 1) o += oyp; else if (cy(a) == -1) o += oym;
    if (cz(a) == 1) o += ozp; else if (cz(a) == -1) o += ozm;
    d[a] = phi[i + o] - pc;
  }
  const T s1 = ((d[1] + d[2]) + (d[3] + d[4])) + (d[5] + d[6]);
  const T s2 = (((d[7] + d[8]) + (d[9] + d[10])) + ((d[11] + d[12]) + (d[13] + d[14]))) + ((d[15] + d[16]) + (d[17] + d[18]));
  L = T(6) * (T(1.0 / 18.0) * s1 + T(1.0 / 36.0) * s2);
  G[0] = T(3) * (T(1.0 / 18.0) * (d[1] - d[2]) + T(1.0 / 36.0) * (((d[7] - d[8]) + (d[9] - d[10])) + ((d[11] - d[12]) + (d[13] - d[14]))));
  G[1] = T(3) * (T(1.0 / 18.0) * (d[3] - d[4]) + T(1.0 / 36.0) * (((d[7] - d[8]) - (d[9] - d[10])) + ((d[15] - d[16]) + (d[17] - d[18]))));
  G[2] = T(3) * (T(1.0 / 18.0) * (d[5] - d[6]) + T(1.0 / 36.0) * (((d[11] - d[12]) - (d[13] - d[14])) + ((d[15] - d[16]) - (d[17] - d[18]))));
}

// ------------------------------------------------------------------------------------------------ physics
template <typename T> struct Mat {  // material state of a node from phi and its stencils
  T rho, inv_rho, tau, s_nu, mu;
};
template <typename T> __device__ __forceinline__ Mat<T> materials(const KP<T>& P, T phi, T L) {
  Mat<T> m;
  m.rho = P.rho_l + phi * P.drho;                                              // Eq. 39
  m.inv_rho = T(1) / m.rho;
  if (P.visc_interp == 1) m.tau = T(1) / (P.itau_l + phi * (P.itau_h - P.itau_l));
  else if (P.visc_interp == 2) m.tau = (P.rt_l + phi * (P.rt_h - P.rt_l)) * m.inv_rho;  // Eq. 25: mu linear, tau = 3 mu / rho
  else m.tau = P.tau_l + phi * (P.tau_h - P.tau_l);                            // Eq. 24
  m.s_nu = T(1) / (m.tau + T(0.5));                                            // G3
  m.mu = P.beta4 * phi * (phi - T(1)) * (phi - T(0.5)) - P.kappa * L;          // Eq. 11 (sign corrected, G4)
  return m;
}

template <typename T> struct Mom {  // p* = sum f, m = sum f e, Pi = sum f e e
  T p, mx, my, mz, xx, yy, zz, xy, yz, xz;
};
template <typename T> __device__ __forceinline__ Mom<T> moments(const T (&f)[Q]) {
  Mom<T> m;
  // pairwise sums / differences of opposite directions
  const T s12 = f[1] + f[2], s34 = f[3] + f[4], s56 = f[5] + f[6];
  const T s78 = f[7] + f[8], s910 = f[9] + f[10], s1112 = f[11] + f[12], s1314 = f[13] + f[14];
  const T s1516 = f[15] + f[16], s1718 = f[17] + f[18];
  const T d12 = f[1] - f[2], d34 = f[3] - f[4], d56 = f[5] - f[6];
  const T d78 = f[7] - f[8], d910 = f[9] - f[10], d1112 = f[11] - f[12], d1314 = f[13] - f[14];
  const T d1516 = f[15] - f[16], d1718 = f[17] - f[18];
  const T sxy = s78 + s910, sxz = s1112 + s1314, syz = s1516 + s1718;
  m.p = (f[0] + (s12 + s34 + s56)) + (sxy + sxz + syz);
  m.mx = d12 + (d78 + d910) + (d1112 + d1314);
  m.my = d34 + (d78 - d910) + (d1516 + d1718);
  m.mz = d56 + (d1112 - d1314) + (d1516 - d1718);
  m.xx = s12 + sxy + sxz;
  m.yy = s34 + sxy + syz;
  m.zz = s56 + sxz + syz;
  m.xy = s78 - s910;
  m.xz = s1112 - s1314;
  m.yz = s1516 - s1718;
  return m;
}

// Total force, Eq. 20: F_s (Eq. 10) + F_b (G16) + F_p (Eq. 21) + F_mu (Eq. 30 in closed form).  Also returns
// D = dev(Pi^neq) for the collision.
template <typename T>
__device__ __forceinline__ void total_force(const KP<T>& P, const Mom<T>& m, const Mat<T>& mat, T ux, T uy, T uz,
                                            const T (&G)[3], T (&F)[3], T (&D)[6]) {
  const T p3 = m.p * T(1.0 / 3.0);
  const T nxx = m.xx - (p3 + ux * ux), nyy = m.yy - (p3 + uy * uy), nzz = m.zz - (p3 + uz * uz);
  const T nxy = m.xy - ux * uy, nyz = m.yz - uy * uz, nxz = m.xz - ux * uz;
  const T tr3 = (nxx + nyy + nzz) * T(1.0 / 3.0);
  D[0] = nxx - tr3; D[1] = nyy - tr3; D[2] = nzz - tr3; D[3] = nxy; D[4] = nyz; D[5] = nxz;
  const T s = mat.s_nu;
  const T trs = P.collision == 1 ? s * tr3 : tr3;  // BGK relaxes the trace at s_nu too (Eq. 29); WMRT at rate 1 (Eq. 30)
  const T Sxx = s * D[0] + trs, Syy = s * D[1] + trs, Szz = s * D[2] + trs;
  const T Sxy = s * D[3], Syz = s * D[4], Sxz = s * D[5];
  const T cmu = -mat.tau * P.drho;
  const T cs = mat.mu - p3 * P.drho;  // F_s + F_p = (mu_phi - p* c_s^2 (rho_h - rho_l)) grad phi
  const T rb = mat.rho - P.rho_ref;
  F[0] = cs * G[0] + rb * P.gx + cmu * (Sxx * G[0] + Sxy * G[1] + Sxz * G[2]);
  F[1] = cs * G[1] + rb * P.gy + cmu * (Sxy * G[0] + Syy * G[1] + Syz * G[2]);
  F[2] = cs * G[2] + rb * P.gz + cmu * (Sxz * G[0] + Syz * G[1] + Szz * G[2]);
}

// Both collisions of one node (Alg. 1): in f, g pre-collision; out post-collision in place.
// PLAIN: the caller guarantees WMRT collision and the full two-phase mode (no runtime mode tests inside the direction loop)
template <typename T, bool PLAIN = false>
__device__ __forceinline__ void collide(const KP<T>& P, const Mom<T>& m, const Mat<T>& mat, T phi, const T (&G)[3], T ux,
                                        T uy, T uz, T (&f)[Q], T (&g)[Q]) {
  T F[3] = {T(0), T(0), T(0)}, D[6] = {T(0), T(0), T(0), T(0), T(0), T(0)};
  if (PLAIN || !P.phase_only) total_force(P, m, mat, ux, uy, uz, G, F, D);
  const T usq15 = T(1.5) * (ux * ux + uy * uy + uz * uz);
  const T hx = T(1.5) * F[0] * mat.inv_rho, hy = T(1.5) * F[1] * mat.inv_rho, hz = T(1.5) * F[2] * mat.inv_rho;
  const T k = T(4.5) * (T(1) - mat.s_nu);
  // interface normal (R10) and F^phi prefactor, Eq. 34
  const T gn = sqrt_(G[0] * G[0] + G[1] * G[1] + G[2] * G[2]) + T(1e-32);
  const T ign = T(1) / gn;
  const T pref = (T(1) - T(4) * (phi - T(0.5)) * (phi - T(0.5))) * P.inv_W;
  const T om = P.om_phi;
  const T cphi = (T(1) - T(0.5) * om) * pref;
  const T nx_ = G[0] * ign * cphi, ny_ = G[1] * ign * cphi, nz_ = G[2] * ign * cphi;
  const T omphi = om * phi, om1 = T(1) - om;
#pragma unroll
  for (int a = 0; a < Q; ++a) {
    const T ex = T(cx(a)), ey = T(cy(a)), ez = T(cz(a));
    const T eu = ex * ux + ey * uy + ez * uz;
    const T gam = T(3) * eu + T(4.5) * eu * eu - usq15;  // Gamma_a / w_a - 1
    const T eDe = ex * ex * D[0] + ey * ey * D[1] + ez * ez * D[2] + T(2) * (ex * ey * D[3] + ey * ez * D[4] + ex * ez * D[5]);
    if (!PLAIN && P.phase_only)  // prescribed u (Sec. 5.4): the hydrodynamic populations are not advanced
      f[a] = T(0);
    else if (!PLAIN && P.collision == 1)  // BGK, Eq. 26: f+ = (1 - s) f + s feq_bar + F_a
      f[a] = (T(1) - mat.s_nu) * f[a] + cw<T>(a) * (mat.s_nu * (m.p + gam) + (T(2) - mat.s_nu) * (ex * hx + ey * hy + ez * hz));
    else
      f[a] = cw<T>(a) * ((m.p + gam) + (ex * hx + ey * hy + ez * hz) + k * eDe);
    g[a] = om1 * g[a] + cw<T>(a) * (omphi * (T(1) + gam) + (ex * nx_ + ey * ny_ + ez * nz_));
  }
}

template <typename T, int a = 0> struct StoreAll {
  static __device__ __forceinline__ void run(T* __restrict__ dst, int nx, long long pb, const T (&v)[Q]) {
    dst[pb + a * nx] = v[a];
    StoreAll<T, a + 1>::run(dst, nx, pb, v);
  }
};
template <typename T> struct StoreAll<T, Q> {
  static __device__ __forceinline__ void run(T* __restrict__, int, long long, const T (&)[Q]) {}
};

// ------------------------------------------------------------------------------------------------ kernels
// lambda = U dt/dy of B.25 for the step t -> t+1, one entry per column of the outlet layer.  U is the
// normal velocity of layer N-1 (B.22, :1104): the stored u_z(x,y,N-1,t) (outlet_u_time = 0, ":1107 previous time step") or the
// first moment of the post-stream f of that layer at t+1 (outlet_u_time = 1, ":1117 after the streaming step"; reading R12).
// U_local: clamped here if outlet_clamp; the plane-wide schemes go on to k_outlet_reduce.
template <typename T> __global__ void __launch_bounds__(256) k_outlet_lam(const __grid_constant__ KP<T> P) {
  const long long c = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= P.nxy) return;
  T U;
  if (P.outlet_u_time == 1 && !P.phase_only) {
    const int x = (int)(c % P.nx), y = (int)(c / P.nx);
    T f[Q], g[Q];
    load_node<T, true, false>(P, x, y, P.nz - 2, f, g);
    U = T(0);
#pragma unroll
    for (int a = 0; a < Q; ++a) if (cz(a) != 0) U += T(cz(a)) * f[a];
  } else {
    U = P.u[2 * P.n + (long long)(P.nz - 2) * P.nxy + c];
  }
  if (P.outlet_u_mode == 0 && P.outlet_clamp && U < T(0)) U = T(0);
  P.lam[c] = U;
}
// Plane-wide outlet velocity of B.22: U_ave (mode 1) or U_max (mode 2) over the per-column values k_outlet_lam
// left in `lam`, clamped at 0 if outlet_clamp, written to every entry.  One block, fixed reduction order (deterministic).
template <typename T> __global__ void __launch_bounds__(1024) k_outlet_reduce(const __grid_constant__ KP<T> P) {
  __shared__ T sh[1024];
  const T* __restrict__ uz = P.lam;
  const bool ave = P.outlet_u_mode == 1;
  T acc = ave ? T(0) : uz[0];
  for (long long c = threadIdx.x; c < P.nxy; c += blockDim.x) {
    const T v = uz[c];
    acc = ave ? acc + v : (v > acc ? v : acc);
  }
  sh[threadIdx.x] = acc;
  __syncthreads();
  for (int s = blockDim.x / 2; s > 0; s >>= 1) {
    if ((int)threadIdx.x < s) {
      const T a = sh[threadIdx.x], b = sh[threadIdx.x + s];
      sh[threadIdx.x] = ave ? a + b : (b > a ? b : a);
    }
    __syncthreads();
  }
  T U = ave ? sh[0] / T(P.nxy) : sh[0];
  if (P.outlet_clamp && U < T(0)) U = T(0);
  __syncthreads();
  for (long long c = threadIdx.x; c < P.nxy; c += blockDim.x) P.lam[c] = U;
}

// k_phi: phi(t+1) = sum_a g_a(x,t+1)  (Eq. 38) from the post-collision g+(t); inlet nodes get phi_in.
template <typename T> __global__ void __launch_bounds__(256) k_phi(const __grid_constant__ KP<T> P) {
  const long long j = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (j >= P.z_cnt * P.nxy) return;
  const long long i = j + (P.z_lo + (P.z_skip && j >= P.z_skip_at * P.nxy ? P.z_skip : 0)) * P.nxy;
  const int x = (int)(i % P.nx);
  const long long r = i / P.nx;
  const int y = (int)(r % P.ny), z = (int)(r / P.ny);
  T f[Q], g[Q];
  load_node<T, false>(P, x, y, z, f, g);
  T s = ((g[0] + (g[1] + g[2])) + ((g[3] + g[4]) + (g[5] + g[6]))) +
        (((g[7] + g[8]) + (g[9] + g[10])) + ((g[11] + g[12]) + (g[13] + g[14])) + ((g[15] + g[16]) + (g[17] + g[18])));
  if (P.has_inlet && z == 0 && P.mask[(long long)y * P.nx + x]) s = P.phi_in;
  P.phi[i] = s;
}

// k_step: the fused stream -> BC -> macro -> collide kernel.
template <typename T, bool PLAIN = false> __global__ void __launch_bounds__(256) k_step(const __grid_constant__ KP<T> P) {
  const long long j = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (j >= P.z_cnt * P.nxy) return;
  const long long i = j + (P.z_lo + (P.z_skip && j >= P.z_skip_at * P.nxy ? P.z_skip : 0)) * P.nxy;
  const int x = (int)(i % P.nx);
  const long long r = i / P.nx;
  const int y = (int)(r % P.ny), z = (int)(r / P.ny);
  T f[Q], g[Q];
  load_node<T, true>(P, x, y, z, f, g);
  if (P.has_outlet && z == P.nz - 1) {  // keep chi(N, t+1) for the next step's B.26-B.27
    const long long c = (long long)y * P.nx + x;
#pragma unroll
    for (int a = 0; a < Q; ++a) { P.ob_f[a * P.nxy + c] = f[a]; P.ob_g[a * P.nxy + c] = g[a]; }
  }
  const T phi = P.phi[i];
  T G[3], L;
  phi_stencil(P, P.phi, x, y, z, phi, G, L);
  const Mat<T> mat = materials(P, phi, L);
  const Mom<T> m = moments(f);
  // macros, Alg. 3: F from (new p*, new phi, lagged u), then Eq. 31b
  T ux = P.u[i], uy = P.u[P.n + i], uz = P.u[2 * P.n + i];
  if (PLAIN || !P.phase_only) {
    T F[3], D[6];
    total_force(P, m, mat, ux, uy, uz, G, F, D);
    const T h = T(0.5) * mat.inv_rho;
    ux = m.mx + h * F[0]; uy = m.my + h * F[1]; uz = m.mz + h * F[2];
  }
  if (P.has_inlet && z == 0 && P.mask[(long long)y * P.nx + x]) { ux = P.uin[0]; uy = P.uin[1]; uz = P.uin[2]; }
  P.u[i] = ux; P.u[P.n + i] = uy; P.u[2 * P.n + i] = uz;
  collide<T, PLAIN>(P, m, mat, phi, G, ux, uy, uz, f, g);
  StoreAll<T>::run(P.p_dst, P.nx, pop_base(i, x), f);
  StoreAll<T>::run(P.p_dst + Q * P.nx, P.nx, pop_base(i, x), g);
}

// k_init: I1-I4 of DESIGN.md (R8), then the first collision; phi0/u0 are caller buffers.
template <typename T>
__global__ void __launch_bounds__(256) k_init(const __grid_constant__ KP<T> P, const T* __restrict__ phi0,
                                              const T* __restrict__ u0) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= P.n) return;
  const int x = (int)(i % P.nx);
  const long long r = i / P.nx;
  const int y = (int)(r % P.ny), z = (int)(r / P.ny);
  const T phi = phi0[i];
  const T ux = u0[i], uy = u0[P.n + i], uz = u0[2 * P.n + i];
  T G[3], L;
  phi_stencil(P, phi0, x, y, z, phi, G, L);
  const Mat<T> mat = materials(P, phi, L);
  // I3: F = F_s + F_b (p* = 0 => F_p = 0; F_mu = 0)
  const T rb = mat.rho - P.rho_ref;
  const T F0 = mat.mu * G[0] + rb * P.gx, F1 = mat.mu * G[1] + rb * P.gy, F2 = mat.mu * G[2] + rb * P.gz;
  const T usq15 = T(1.5) * (ux * ux + uy * uy + uz * uz);
  const T gn = sqrt_(G[0] * G[0] + G[1] * G[1] + G[2] * G[2]) + T(1e-32);
  const T pref = (T(1) - T(4) * (phi - T(0.5)) * (phi - T(0.5))) * P.inv_W / gn;
  T f[Q], g[Q];
#pragma unroll
  for (int a = 0; a < Q; ++a) {
    const T ex = T(cx(a)), ey = T(cy(a)), ez = T(cz(a));
    const T eu = ex * ux + ey * uy + ez * uz;
    const T gam = T(3) * eu + T(4.5) * eu * eu - usq15;
    const T Fa = T(3) * (ex * F0 + ey * F1 + ez * F2) * mat.inv_rho;  // Eq. 19 / w_a
    const T Fp = pref * (ex * G[0] + ey * G[1] + ez * G[2]);          // Eq. 34 / w_a
    f[a] = cw<T>(a) * (gam - T(0.5) * Fa);                            // I4
    g[a] = cw<T>(a) * (phi * (T(1) + gam) - T(0.5) * Fp);
  }
  if (P.has_outlet && z == P.nz - 1) {
    const long long c = (long long)y * P.nx + x;
#pragma unroll
    for (int a = 0; a < Q; ++a) { P.ob_f[a * P.nxy + c] = f[a]; P.ob_g[a * P.nxy + c] = g[a]; }
  }
  P.phi[i] = phi;
  P.u[i] = ux; P.u[P.n + i] = uy; P.u[2 * P.n + i] = uz;
  const Mom<T> m = moments(f);
  collide(P, m, mat, phi, G, ux, uy, uz, f, g);
  StoreAll<T>::run(P.p_dst, P.nx, pop_base(i, x), f);
  StoreAll<T>::run(P.p_dst + Q * P.nx, P.nx, pop_base(i, x), g);
}

// k_get: phi, p = p* rho c_s^2 with p* = sum_a f+_a (the collision conserves sum f), u.
template <typename T>
__global__ void __launch_bounds__(256) k_get(const __grid_constant__ KP<T> P, T* __restrict__ phi_out, T* __restrict__ p_out,
                                             T* __restrict__ u_out) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= P.n) return;
  const T phi = P.phi[i];
  if (phi_out) phi_out[i] = phi;
  if (u_out) { u_out[i] = P.u[i]; u_out[P.n + i] = P.u[P.n + i]; u_out[2 * P.n + i] = P.u[2 * P.n + i]; }
  if (p_out) {
    T f[Q];
    const int x = (int)(i % P.nx);
#pragma unroll
    for (int a = 0; a < Q; ++a) f[a] = P.p_src[pop_base(i, x) + a * P.nx];
    const Mom<T> m = moments(f);
    p_out[i] = m.p * (P.rho_l + phi * P.drho) * T(1.0 / 3.0);
  }
}

}  // namespace clip
