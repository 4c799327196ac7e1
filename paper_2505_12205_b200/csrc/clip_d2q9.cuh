// clip_d2q9.cuh -- the same time step on the D2Q9 lattice, the lattice of the paper's 2-D benchmarks ("For 2D
// problems, the D2Q9 lattice model is utilized"; capillary wave :570-596, layered Poiseuille :647-669, interface in shear flow
// :675-713; Table 2 :561 times a 256 x 64 D2Q9 case).  Equations, readings and the lean arithmetic are those of clip_kernels.cuh with
// the two-dimensional velocity set: weights 4/9, 1/9, 1/36, c_s^2 = 1/3, and the TWO traceless second-order moments
// {e_x e_y, e_x^2 - e_y^2} relaxing at s_nu (G2 in two dimensions), so that
//   M^-1 S M = I - (1 - s_nu) P,  P_ab = w_a / (2 c_s^4) Q_a : dev2(Q_b),  dev2 = traceless part of a 2 x 2 tensor
//   f+_a = w_a [p* + 3 e.u + 4.5 (e.u)^2 - 1.5 u.u + 1.5 e.F / rho + 4.5 (1 - s_nu) e^T D e],  D = dev2(Pi^neq)
//   F_mu = -tau (rho_h - rho_l) [s_nu D + tr(Pi^neq)/2 I] . grad phi   (BGK: s_nu on the trace as well, Eq. 29)
// Thread per node, scalar, two kernels per step (k_phi9: phi(t+1) = sum_a g_a after streaming; k_step9: the rest), the design "D0"
// of DESIGN.md: 2-D lattices are small, the 3-D lattices carry the throughput work.  Faces: PERIODIC, WALL (halfway bounce-back),
// FREESLIP in x and y; nz = 1.  State: pop [ny][18][nx] (A/B), phi [ny][nx], u [3][ny][nx] (u_z == 0, never touched by a step).
#pragma once
#include "clip_kernels.cuh"
#include "clip_fused.cuh"
#include <type_traits>

namespace clip {
namespace d2q9 {

constexpr int Q9 = 9;
constexpr int NC9 = 2 * Q9;
// rest; (+-1, 0); (0, +-1); (1,1), (-1,-1); (1,-1), (-1,1): opposite directions adjacent (a odd -> a + 1)
__host__ __device__ constexpr int ex(int a) { return (a == 1 || a == 5 || a == 7) ? 1 : ((a == 2 || a == 6 || a == 8) ? -1 : 0); }
__host__ __device__ constexpr int ey(int a) { return (a == 3 || a == 5 || a == 8) ? 1 : ((a == 4 || a == 6 || a == 7) ? -1 : 0); }
__host__ __device__ constexpr int opp9(int a) { return a == 0 ? 0 : ((a & 1) ? a + 1 : a - 1); }
template <typename T> __host__ __device__ constexpr T w9(int a) { return a == 0 ? T(4.0 / 9.0) : (a < 5 ? T(1.0 / 9.0) : T(1.0 / 36.0)); }
__host__ __device__ constexpr int dir9(int x, int y) {
  for (int a = 0; a < Q9; ++a) if (ex(a) == x && ey(a) == y) return a;
  return 0;
}

__device__ __forceinline__ long long pidx(int nx, int y, int c, int x) { return ((long long)y * NC9 + c) * nx + x; }

// Streaming (pull; Alg. 2, B.3-B.6) of direction a of set `set` (0: f, 1: g) at node (x, y): periodic wrap, halfway bounce-back
// (B.10-B.11; a wall crossing wins at corners, R11), specular reflection at free-slip faces (B.8-B.9, pull form).
template <typename T, int a> __device__ __forceinline__ T pull9(const KP<T>& P, int set, int x, int y) {
  const T* __restrict__ src = P.p_src;
  if (a == 0) return __ldg(src + pidx(P.nx, y, set * Q9, x));
  int sx = x - ex(a), sy = y - ey(a), fx = ex(a), fy = ey(a);
  bool bounce = false;
  if (ex(a) != 0 && (sx < 0 || sx >= P.nx)) {
    const int bc = P.bc[sx < 0 ? 0 : 1];
    if (bc == BC_PERIODIC) sx = sx < 0 ? P.nx - 1 : 0;
    else if (bc == BC_FREESLIP) { sx = x; fx = -fx; }
    else bounce = true;
  }
  if (ey(a) != 0 && (sy < 0 || sy >= P.ny)) {
    const int bc = P.bc[sy < 0 ? 2 : 3];
    if (bc == BC_PERIODIC) sy = sy < 0 ? P.ny - 1 : 0;
    else if (bc == BC_FREESLIP) { sy = y; fy = -fy; }
    else bounce = true;
  }
  if (bounce) return __ldg(src + pidx(P.nx, y, set * Q9 + opp9(a), x));
  const int as = (fx == ex(a) && fy == ey(a)) ? a : dir9(fx, fy);
  return __ldg(src + pidx(P.nx, sy, set * Q9 + as, sx));
}
template <typename T, int a = 0> struct Pull9 {
  static __device__ __forceinline__ void run(const KP<T>& P, int set, int x, int y, T (&v)[Q9]) {
    v[a] = pull9<T, a>(P, set, x, y);
    Pull9<T, a + 1>::run(P, set, x, y, v);
  }
};
template <typename T> struct Pull9<T, Q9> { static __device__ __forceinline__ void run(const KP<T>&, int, int, int, T (&)[Q9]) {} };

// Eq. 40a/b with the D2Q9 weights on differences d_a = phi(x + e_a) - phi(x); ghost rule: wrap or clamp (R9)
template <typename T> __device__ __forceinline__ void stencil9(const KP<T>& P, const T* __restrict__ phi, int x, int y, T pc, T (&G)[3], T& L) {
  const int xm = x > 0 ? x - 1 : (P.bc[0] == BC_PERIODIC ? P.nx - 1 : 0), xp = x < P.nx - 1 ? x + 1 : (P.bc[1] == BC_PERIODIC ? 0 : P.nx - 1);
  const int ym = y > 0 ? y - 1 : (P.bc[2] == BC_PERIODIC ? P.ny - 1 : 0), yp = y < P.ny - 1 ? y + 1 : (P.bc[3] == BC_PERIODIC ? 0 : P.ny - 1);
  const T* __restrict__ r0 = phi + (long long)y * P.nx;
  const T* __restrict__ rm = phi + (long long)ym * P.nx;
  const T* __restrict__ rp = phi + (long long)yp * P.nx;
  const T d1 = r0[xp] - pc, d2 = r0[xm] - pc, d3 = rp[x] - pc, d4 = rm[x] - pc;
  const T d5 = rp[xp] - pc, d6 = rm[xm] - pc, d7 = rm[xp] - pc, d8 = rp[xm] - pc;
  L = T(6) * (T(1.0 / 9.0) * ((d1 + d2) + (d3 + d4)) + T(1.0 / 36.0) * ((d5 + d6) + (d7 + d8)));
  G[0] = T(3) * (T(1.0 / 9.0) * (d1 - d2) + T(1.0 / 36.0) * ((d5 - d6) + (d7 - d8)));
  G[1] = T(3) * (T(1.0 / 9.0) * (d3 - d4) + T(1.0 / 36.0) * ((d5 - d6) - (d7 - d8)));
  G[2] = T(0);
}

template <typename T> struct Mom9 { T p, mx, my, xx, yy, xy; };
template <typename T> __device__ __forceinline__ Mom9<T> moments9(const T (&f)[Q9]) {
  Mom9<T> m;
  const T s12 = f[1] + f[2], s34 = f[3] + f[4], s56 = f[5] + f[6], s78 = f[7] + f[8];
  const T d12 = f[1] - f[2], d34 = f[3] - f[4], d56 = f[5] - f[6], d78 = f[7] - f[8];
  m.p = (f[0] + (s12 + s34)) + (s56 + s78);
  m.mx = d12 + (d56 + d78);
  m.my = d34 + (d56 - d78);
  m.xx = s12 + (s56 + s78);
  m.yy = s34 + (s56 + s78);
  m.xy = s56 - s78;
  return m;
}
// Total force (Eq. 20) and D = dev2(Pi^neq) = (Dxx, Dxy), Dyy = -Dxx
template <typename T>
__device__ __forceinline__ void force9(const KP<T>& P, const Mom9<T>& m, const Mat<T>& mat, T ux, T uy, const T (&G)[3], T (&F)[2], T (&D)[2]) {
  const T p3 = m.p * T(1.0 / 3.0);
  const T nxx = m.xx - (p3 + ux * ux), nyy = m.yy - (p3 + uy * uy), nxy = m.xy - ux * uy;
  const T tr2 = T(0.5) * (nxx + nyy);
  D[0] = nxx - tr2; D[1] = nxy;
  const T s = mat.s_nu;
  const T trs = P.collision == 1 ? s * tr2 : tr2;   // BGK relaxes the trace at s_nu too (Eq. 29); WMRT at rate 1 (Eq. 30)
  const T Sxx = s * D[0] + trs, Syy = trs - s * D[0], Sxy = s * D[1];
  const T cmu = -mat.tau * P.drho;
  const T cs = mat.mu - p3 * P.drho;                 // F_s + F_p
  const T rb = mat.rho - P.rho_ref;
  F[0] = cs * G[0] + rb * P.gx + cmu * (Sxx * G[0] + Sxy * G[1]);
  F[1] = cs * G[1] + rb * P.gy + cmu * (Sxy * G[0] + Syy * G[1]);
}
// Both collisions of one node (Alg. 1): in f, g pre-collision; out post-collision in place.
template <typename T>
__device__ __forceinline__ void collide9(const KP<T>& P, const Mom9<T>& m, const Mat<T>& mat, T phi, const T (&G)[3], T ux, T uy,
                                         T (&f)[Q9], T (&g)[Q9]) {
  T F[2] = {T(0), T(0)}, D[2] = {T(0), T(0)};
  if (!P.phase_only) force9(P, m, mat, ux, uy, G, F, D);
  const T usq15 = T(1.5) * (ux * ux + uy * uy);
  const T hx = T(1.5) * F[0] * mat.inv_rho, hy = T(1.5) * F[1] * mat.inv_rho;
  const T k = T(4.5) * (T(1) - mat.s_nu);
  const T gn = sqrt_(G[0] * G[0] + G[1] * G[1]) + T(1e-32);   // R10
  const T pref = (T(1) - T(4) * (phi - T(0.5)) * (phi - T(0.5))) * P.inv_W;
  const T om = P.om_phi;
  const T cphi = (T(1) - T(0.5) * om) * pref / gn;
  const T nx_ = G[0] * cphi, ny_ = G[1] * cphi;
  const T omphi = om * phi, om1 = T(1) - om;
#pragma unroll
  for (int a = 0; a < Q9; ++a) {
    const T cx_ = T(ex(a)), cy_ = T(ey(a));
    const T eu = cx_ * ux + cy_ * uy;
    const T gam = T(3) * eu + T(4.5) * eu * eu - usq15;
    const T eDe = (cx_ * cx_ - cy_ * cy_) * D[0] + T(2) * cx_ * cy_ * D[1];
    if (P.phase_only) f[a] = T(0);
    else if (P.collision == 1) f[a] = (T(1) - mat.s_nu) * f[a] + w9<T>(a) * (mat.s_nu * (m.p + gam) + (T(2) - mat.s_nu) * (cx_ * hx + cy_ * hy));
    else f[a] = w9<T>(a) * ((m.p + gam) + (cx_ * hx + cy_ * hy) + k * eDe);
    g[a] = om1 * g[a] + w9<T>(a) * (omphi * (T(1) + gam) + (cx_ * nx_ + cy_ * ny_));
  }
}
template <typename T> __device__ __forceinline__ void store9(const KP<T>& P, int x, int y, const T (&f)[Q9], const T (&g)[Q9]) {
#pragma unroll
  for (int a = 0; a < Q9; ++a) { P.p_dst[pidx(P.nx, y, a, x)] = f[a]; P.p_dst[pidx(P.nx, y, Q9 + a, x)] = g[a]; }
}

template <typename T> __global__ void __launch_bounds__(256) k_phi9(const __grid_constant__ KP<T> P) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= P.n) return;
  const int x = (int)(i % P.nx), y = (int)(i / P.nx);
  T g[Q9];
  Pull9<T>::run(P, 1, x, y, g);
  P.phi[i] = (g[0] + ((g[1] + g[2]) + (g[3] + g[4]))) + ((g[5] + g[6]) + (g[7] + g[8]));
}
template <typename T> __global__ void __launch_bounds__(256) k_step9(const __grid_constant__ KP<T> P) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= P.n) return;
  const int x = (int)(i % P.nx), y = (int)(i / P.nx);
  T f[Q9], g[Q9];
  Pull9<T>::run(P, 0, x, y, f);
  Pull9<T>::run(P, 1, x, y, g);
  const T phi = P.phi[i];
  T G[3], L;
  stencil9(P, P.phi, x, y, phi, G, L);
  const Mat<T> mat = materials(P, phi, L);
  const Mom9<T> m = moments9(f);
  T ux = P.u[i], uy = P.u[P.n + i];
  if (!P.phase_only) {  // macros, Alg. 3: F from (new p*, new phi, lagged u, R13), then Eq. 31b
    T F[2], D[2];
    force9(P, m, mat, ux, uy, G, F, D);
    const T h = T(0.5) * mat.inv_rho;
    ux = m.mx + h * F[0]; uy = m.my + h * F[1];
    P.u[i] = ux; P.u[P.n + i] = uy;
  }
  collide9(P, m, mat, phi, G, ux, uy, f, g);
  store9(P, x, y, f, g);
}
// I1-I4 of DESIGN.md (R8), then the first collision
template <typename T> __global__ void __launch_bounds__(256) k_init9(const __grid_constant__ KP<T> P, const T* __restrict__ phi0, const T* __restrict__ u0) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= P.n) return;
  const int x = (int)(i % P.nx), y = (int)(i / P.nx);
  const T phi = phi0[i], ux = u0[i], uy = u0[P.n + i];
  T G[3], L;
  stencil9(P, phi0, x, y, phi, G, L);
  const Mat<T> mat = materials(P, phi, L);
  const T rb = mat.rho - P.rho_ref;
  const T F0 = mat.mu * G[0] + rb * P.gx, F1 = mat.mu * G[1] + rb * P.gy;   // I3: F = F_s + F_b (p* = 0, F_mu = 0)
  const T usq15 = T(1.5) * (ux * ux + uy * uy);
  const T gn = sqrt_(G[0] * G[0] + G[1] * G[1]) + T(1e-32);
  const T pref = (T(1) - T(4) * (phi - T(0.5)) * (phi - T(0.5))) * P.inv_W / gn;
  T f[Q9], g[Q9];
#pragma unroll
  for (int a = 0; a < Q9; ++a) {
    const T cx_ = T(ex(a)), cy_ = T(ey(a));
    const T eu = cx_ * ux + cy_ * uy;
    const T gam = T(3) * eu + T(4.5) * eu * eu - usq15;
    f[a] = P.phase_only ? T(0) : w9<T>(a) * (gam - T(0.5) * (T(3) * (cx_ * F0 + cy_ * F1) * mat.inv_rho));   // I4
    g[a] = w9<T>(a) * (phi * (T(1) + gam) - T(0.5) * (pref * (cx_ * G[0] + cy_ * G[1])));
  }
  P.phi[i] = phi;
  P.u[i] = ux; P.u[P.n + i] = uy; P.u[2 * P.n + i] = T(0);
  const Mom9<T> m = moments9(f);
  collide9(P, m, mat, phi, G, ux, uy, f, g);
  store9(P, x, y, f, g);
}
// phi, p = p* rho c_s^2 with p* = sum_a f+_a, u
template <typename T>
__global__ void __launch_bounds__(256) k_get9(const __grid_constant__ KP<T> P, T* __restrict__ phi_out, T* __restrict__ p_out, T* __restrict__ u_out) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= P.n) return;
  const int x = (int)(i % P.nx), y = (int)(i / P.nx);
  const T phi = P.phi[i];
  if (phi_out) phi_out[i] = phi;
  if (u_out) { u_out[i] = P.u[i]; u_out[P.n + i] = P.u[P.n + i]; u_out[2 * P.n + i] = P.u[2 * P.n + i]; }
  if (p_out) {
    T f[Q9];
#pragma unroll
    for (int a = 0; a < Q9; ++a) f[a] = P.p_src[pidx(P.nx, y, a, x)];
    p_out[i] = moments9(f).p * (P.rho_l + phi * P.drho) * T(1.0 / 3.0);
  }
}

}  // namespace d2q9
}  // namespace clip

// ------------------------------------------------------------------------------------------------------------------------------
// Pair-per-thread D2Q9 kernels (even nx): one thread owns the node pair (x0, x0 + 1) of a row, two-lane packed arithmetic
// (clip_pack.cuh: FFMA2 / FADD2 / FMUL2 in fp32), every wrap / bounce-back / free-slip case SELECTS the address of a load (as pull2 of
// clip_fast.cuh).  Same two-kernel step as k_phi9 + k_step9; odd nx and `path = 1` keep the scalar kernels.
#include "clip_pack.cuh"

namespace clip {
namespace d2q9 {

struct Geo9 {
  int x0, nx;
  long long r0, rm, rp;     // population-row starts (element index of component 0, column 0) of the rows y, y-1, y+1 (periodic wrap)
  int p0, pm, pp;           // phi-row starts of y and of the ghost-rule rows y-1, y+1 (wrap or clamp)
  bool wm, wp;              // x0-1 / x0+2 wrap around
  bool bxm, bxp, bym, byp;  // links that cross a WALL face
  bool sxm, sxp, sym, syp;  // links that cross a FREESLIP face
  int cxm, cxp;             // phi column offsets from x0 to x0-1 and x0+2 under the ghost rule
};
template <typename T> __device__ __forceinline__ Geo9 make_geo9(const KP<T>& P, int x0, int y) {
  Geo9 g;
  g.x0 = x0; g.nx = P.nx;
  const int ym = y > 0 ? y - 1 : P.ny - 1, yp = y < P.ny - 1 ? y + 1 : 0;
  g.r0 = (long long)y * NC9 * P.nx; g.rm = (long long)ym * NC9 * P.nx; g.rp = (long long)yp * NC9 * P.nx;
  g.wm = x0 == 0; g.wp = x0 + 2 == P.nx;
  g.bxm = g.wm && P.bc[0] == BC_WALL; g.sxm = g.wm && P.bc[0] == BC_FREESLIP;
  g.bxp = g.wp && P.bc[1] == BC_WALL; g.sxp = g.wp && P.bc[1] == BC_FREESLIP;
  g.bym = y == 0 && P.bc[2] == BC_WALL; g.sym = y == 0 && P.bc[2] == BC_FREESLIP;
  g.byp = y == P.ny - 1 && P.bc[3] == BC_WALL; g.syp = y == P.ny - 1 && P.bc[3] == BC_FREESLIP;
  g.p0 = y * P.nx;
  g.pm = ((y == 0 && P.bc[2] != BC_PERIODIC) ? y : ym) * P.nx;
  g.pp = ((y == P.ny - 1 && P.bc[3] != BC_PERIODIC) ? y : yp) * P.nx;
  g.cxm = g.wm ? (P.bc[0] == BC_PERIODIC ? P.nx - 1 : 0) : -1;
  g.cxp = g.wp ? (P.bc[1] == BC_PERIODIC ? 2 - P.nx : 1) : 2;
  return g;
}
// LEAN: the pair is away from every face and from the row ends (no wrap, bounce or reflection to select): plain shifted loads
template <typename T, int a, int SET, bool LEAN = false> __device__ __forceinline__ P2<T> pull9p(const T* __restrict__ src, const Geo9& g) {
  const int nx = g.nx;
  const long long rs = ey(a) == 1 ? g.rm : (ey(a) == -1 ? g.rp : g.r0);   // the row the population comes from
  const T* __restrict__ rp = src + rs + (SET * Q9 + a) * nx + g.x0;
  if (a == 0) return ld_pair<T>(rp);
  if (LEAN) {
    if (ex(a) == 0) return ld_pair<T>(rp);
    return ex(a) == 1 ? P2<T>(ld_one<T>(rp - 1), ld_one<T>(rp)) : P2<T>(ld_one<T>(rp + 1), ld_one<T>(rp + 2));
  }
  const T* __restrict__ own = src + g.r0 + (SET * Q9 + opp9(a)) * nx + g.x0;
  const bool rb = (ey(a) == 1 && g.bym) || (ey(a) == -1 && g.byp);
  const bool ry = (ey(a) == 1 && g.sym) || (ey(a) == -1 && g.syp);
  const T* __restrict__ srx = src + rs + (SET * Q9 + dir9(-ex(a), ey(a))) * nx + g.x0;   // x-reflected source
  if (ey(a) != 0 && ry) {
    rp = src + g.r0 + (SET * Q9 + dir9(ex(a), -ey(a))) * nx + g.x0;
    srx = src + g.r0 + (SET * Q9 + dir9(-ex(a), -ey(a))) * nx + g.x0;
  }
  if (ex(a) == 0) return ld_pair<T>(rb ? own : rp);
  const T* __restrict__ plo;
  const T* __restrict__ phi;
  if (ex(a) == 1) {
    plo = rp + (g.wm ? nx - 1 : -1); phi = rp;
    if (g.sxm) plo = srx;
    if (g.bxm) plo = own;
  } else {
    plo = rp + 1; phi = rp + (g.wp ? 2 - nx : 2);
    if (g.sxp) phi = srx + 1;
    if (g.bxp) phi = own + 1;
  }
  if (rb) { plo = own; phi = own + 1; }
  return P2<T>(ld_one<T>(plo), ld_one<T>(phi));
}
template <typename T, int SET, bool LEAN = false, int a = 0> struct Pull9p {
  static __device__ __forceinline__ void run(const T* __restrict__ src, const Geo9& g, P2<T> (&v)[Q9]) {
    v[a] = pull9p<T, a, SET, LEAN>(src, g);
    Pull9p<T, SET, LEAN, a + 1>::run(src, g, v);
  }
};
template <typename T, int SET, bool LEAN> struct Pull9p<T, SET, LEAN, Q9> { static __device__ __forceinline__ void run(const T* __restrict__, const Geo9&, P2<T> (&)[Q9]) {} };

template <typename T> struct Row3p { P2<T> L, C, R; };
template <typename T, bool LEAN = false> __device__ __forceinline__ Row3p<T> ld_row3p(const T* __restrict__ phi, int row, const Geo9& g) {
  Row3p<T> r;
  r.C = ld_pair<T>(phi + row + g.x0);
  const T m = ld_one<T>(phi + row + g.x0 + (LEAN ? -1 : g.cxm)), p = ld_one<T>(phi + row + g.x0 + (LEAN ? 2 : g.cxp));
  r.L = P2<T>(m, r.C.lo());
  r.R = P2<T>(r.C.hi(), p);
  return r;
}
template <typename T, bool LEAN = false> __device__ __forceinline__ void stencil9p(const T* __restrict__ phi, const Geo9& g, P2<T>& pc, P2<T> (&G)[2], P2<T>& L) {
  typedef P2<T> V;
  const Row3p<T> c = ld_row3p<T, LEAN>(phi, g.p0, g), yp = ld_row3p<T, LEAN>(phi, g.pp, g), ym = ld_row3p<T, LEAN>(phi, g.pm, g);
  pc = c.C;
  const V d1 = c.R - pc, d2 = c.L - pc, d3 = yp.C - pc, d4 = ym.C - pc;
  const V d5 = yp.R - pc, d6 = ym.L - pc, d7 = ym.R - pc, d8 = yp.L - pc;
  L = fma2(V(T(6.0 / 9.0)), (d1 + d2) + (d3 + d4), V(T(6.0 / 36.0)) * ((d5 + d6) + (d7 + d8)));
  G[0] = fma2(V(T(3.0 / 9.0)), d1 - d2, V(T(3.0 / 36.0)) * ((d5 - d6) + (d7 - d8)));
  G[1] = fma2(V(T(3.0 / 9.0)), d3 - d4, V(T(3.0 / 36.0)) * ((d5 - d6) - (d7 - d8)));
}

template <typename T> struct Mom9p { P2<T> p, mx, my, xx, yy, xy; };
template <typename T> __device__ __forceinline__ Mom9p<T> moments9p(const P2<T> (&f)[Q9]) {
  typedef P2<T> V;
  Mom9p<T> m;
  const V s12 = f[1] + f[2], s34 = f[3] + f[4], s56 = f[5] + f[6], s78 = f[7] + f[8];
  const V d12 = f[1] - f[2], d34 = f[3] - f[4], d56 = f[5] - f[6], d78 = f[7] - f[8];
  m.p = (f[0] + (s12 + s34)) + (s56 + s78);
  m.mx = d12 + (d56 + d78);
  m.my = d34 + (d56 - d78);
  m.xx = s12 + (s56 + s78);
  m.yy = s34 + (s56 + s78);
  m.xy = s56 - s78;
  return m;
}
template <typename T> struct Mat9p { P2<T> rho, inv_rho, tau, s_nu, mu; };
template <typename T> __device__ __forceinline__ Mat9p<T> materials9p(const KP<T>& P, P2<T> phi, P2<T> L) {
  typedef P2<T> V;
  Mat9p<T> m;
  m.rho = fma2(phi, V(P.drho), V(P.rho_l));
  m.inv_rho = rcp2(m.rho);
  if (P.visc_interp == 1) m.tau = rcp2(fma2(phi, V(P.itau_h - P.itau_l), V(P.itau_l)));
  else if (P.visc_interp == 2) m.tau = fma2(phi, V(P.rt_h - P.rt_l), V(P.rt_l)) * m.inv_rho;
  else m.tau = fma2(phi, V(P.tau_h - P.tau_l), V(P.tau_l));
  m.s_nu = rcp2(m.tau + V(T(0.5)));
  m.mu = fms2(V(P.beta4) * phi, (phi - V(T(1))) * (phi - V(T(0.5))), V(P.kappa) * L);
  return m;
}
template <typename T>
__device__ __forceinline__ void force9p(const KP<T>& P, const Mom9p<T>& m, const Mat9p<T>& mat, P2<T> ux, P2<T> uy, const P2<T> (&G)[2],
                                        P2<T> (&F)[2], P2<T> (&D)[2]) {
  typedef P2<T> V;
  const V p3 = m.p * V(T(1.0 / 3.0));
  const V nxx = m.xx - fma2(ux, ux, p3), nyy = m.yy - fma2(uy, uy, p3), nxy = m.xy - ux * uy;
  const V tr2 = V(T(0.5)) * (nxx + nyy);
  D[0] = nxx - tr2; D[1] = nxy;
  const V s = mat.s_nu;
  const V trs = P.collision == 1 ? s * tr2 : tr2;
  const V Sxx = fma2(s, D[0], trs), Syy = trs - s * D[0], Sxy = s * D[1];
  const V cmu = -(mat.tau * V(P.drho));
  const V cs = mat.mu - p3 * V(P.drho);
  const V rb = mat.rho - V(P.rho_ref);
  F[0] = fma2(cs, G[0], fma2(rb, V(P.gx), cmu * fma2(Sxx, G[0], Sxy * G[1])));
  F[1] = fma2(cs, G[1], fma2(rb, V(P.gy), cmu * fma2(Sxy, G[0], Syy * G[1])));
}
template <typename T>
__device__ __forceinline__ void collide9p(const KP<T>& P, const Mom9p<T>& m, const Mat9p<T>& mat, P2<T> phi, const P2<T> (&G)[2], P2<T> ux,
                                          P2<T> uy, P2<T> (&f)[Q9], P2<T> (&g)[Q9]) {
  typedef P2<T> V;
  V F[2] = {V(T(0)), V(T(0))}, D[2] = {V(T(0)), V(T(0))};
  if (!P.phase_only) force9p(P, m, mat, ux, uy, G, F, D);
  const V usq15 = V(T(1.5)) * fma2(ux, ux, uy * uy);
  const V ir15 = V(T(1.5)) * mat.inv_rho;
  const V hx = F[0] * ir15, hy = F[1] * ir15;
  const V k = V(T(4.5)) * (V(T(1)) - mat.s_nu);
  const V gn = sqrt2(fma2(G[0], G[0], G[1] * G[1])) + V(T(1e-32));
  const V ph = phi - V(T(0.5));
  const V pref = fma2(V(T(-4)) * ph, ph, V(T(1))) * V(P.inv_W);
  const V cphi = (V(T(1) - T(0.5) * P.om_phi) * pref) * rcp2(gn);
  const V nx_ = G[0] * cphi, ny_ = G[1] * cphi;
  const V omphi = V(P.om_phi) * phi, om1 = V(T(1) - P.om_phi);
#pragma unroll
  for (int a = 0; a < Q9; ++a) {
    const V cx_ = V(T(ex(a))), cy_ = V(T(ey(a)));
    const V eu = fma2(cx_, ux, cy_ * uy);
    const V gam = fma2(V(T(4.5)) * eu, eu, fma2(V(T(3)), eu, -usq15));
    const V eDe = fma2(V(T(ex(a) * ex(a) - ey(a) * ey(a))), D[0], V(T(2 * ex(a) * ey(a))) * D[1]);
    const V eh = fma2(cx_, hx, cy_ * hy);
    const V w(w9<T>(a));
    if (P.phase_only) f[a] = V(T(0));
    else if (P.collision == 1) f[a] = fma2(V(T(1)) - mat.s_nu, f[a], w * fma2(mat.s_nu, m.p + gam, (V(T(2)) - mat.s_nu) * eh));
    else f[a] = w * ((m.p + gam) + fma2(k, eDe, eh));
    g[a] = fma2(om1, g[a], w * fma2(omphi, V(T(1)) + gam, fma2(cx_, nx_, cy_ * ny_)));
  }
}
template <typename T> __device__ __forceinline__ bool pair9_coords(const KP<T>& P, int& x0, int& y) {
  x0 = 2 * (blockIdx.x * blockDim.x + threadIdx.x);
  y = blockIdx.y;
  return x0 < P.nx;
}
// grid = (ceil(nx / 2 / blockDim.x), ny)
template <typename T> __global__ void __launch_bounds__(128) k_phi9p(const __grid_constant__ KP<T> P) {
  int x0, y;
  if (!pair9_coords(P, x0, y)) return;
  const Geo9 g = make_geo9(P, x0, y);
  P2<T> v[Q9];
  Pull9p<T, 1>::run(P.p_src, g, v);
  st_pair<T>(P.phi + g.p0 + x0, (v[0] + ((v[1] + v[2]) + (v[3] + v[4]))) + ((v[5] + v[6]) + (v[7] + v[8])));
}
// One node pair of row y: stream -> BC -> macros -> both collisions -> store; g holds the post-collision g+ on return.
template <typename T, bool LEAN = false> __device__ __forceinline__ void step9p_pair(const KP<T>& P, const Geo9& geo, int x0, P2<T> (&g)[Q9]) {
  typedef P2<T> V;
  V f[Q9];
  Pull9p<T, 0, LEAN>::run(P.p_src, geo, f);
  Pull9p<T, 1, LEAN>::run(P.p_src, geo, g);
  const int i = geo.p0 + x0;
  V ux = ld_pair<T>(P.u + i), uy = ld_pair<T>(P.u + P.n + i);
  V phi, G[2], L;
  stencil9p<T, LEAN>(P.phi, geo, phi, G, L);
  const Mat9p<T> mat = materials9p<T>(P, phi, L);
  const Mom9p<T> m = moments9p<T>(f);
  if (!P.phase_only) {  // macros, Alg. 3 (lagged u, R13), then Eq. 31b
    V F[2], D[2];
    force9p(P, m, mat, ux, uy, G, F, D);
    const V h = V(T(0.5)) * mat.inv_rho;
    ux = fma2(h, F[0], m.mx); uy = fma2(h, F[1], m.my);
    st_pair<T>(P.u + i, ux); st_pair<T>(P.u + P.n + i, uy);
  }
  collide9p<T>(P, m, mat, phi, G, ux, uy, f, g);
  T* const rd = P.p_dst + geo.r0 + x0;
#pragma unroll
  for (int a = 0; a < Q9; ++a) { st_pair<T>(rd + a * P.nx, f[a]); st_pair<T>(rd + (Q9 + a) * P.nx, g[a]); }
}
template <typename T> __global__ void __launch_bounds__(128) k_step9p(const __grid_constant__ KP<T> P) {
  int x0, y;
  if (!pair9_coords(P, x0, y)) return;
  const Geo9 geo = make_geo9(P, x0, y);
  P2<T> g[Q9];
  step9p_pair<T>(P, geo, x0, g);
}

// ------------------------------------------------------------------------------------------------ single pass (k_fused9 + k_fix9)
// The 2-D analogue of k_fused (clip_fused.cuh): ONE pass over f and g per step.  A block owns a chunk of whole lattice rows
// [yc[c], yc[c+1]) and walks it row by row, 2 * blockDim.x nodes at a time; phi(t+2) = sum_a g+_a(x - e_a, t+1) is accumulated on chip
// from the g+ just computed, in a shared-memory ring of four rows (y-1, y, y+1 and the one being flushed): the three x-directions of
// a target row are combined by warp shuffles, every thread adds only into its own column pair, what crosses a warp's 64-node column
// group goes through the edge arrays (periodic wrap in x included).  Finished rows are flushed to phi_dst, the two rows just outside
// the chunk to `part` [chunk][2][nx]; k_fix9 adds them to the first / last row of the neighbouring chunks (fixed order, deterministic).
// WALL / FREESLIP faces: where a population lands -- a link through a wall returns to the sender (B.10-B.11), a link through a
// free-slip face keeps its tangential displacement (B.8-B.9), a wall crossing anywhere wins (R11).
constexpr int FUSED9_MAX_CHUNKS = 2048;
template <typename T> struct Fused9P {
  T* phi_dst;   // phi(t+2)                                   [ny][nx]
  T* part;      // the two halo rows of every chunk            [nchunks][2][nx]
  int nchunks;  // chunk c covers the rows c * ny / nchunks .. (c + 1) * ny / nchunks - 1
};
template <typename T> struct Tri9 { P2<T> v0, vp, vm; };

template <typename T>
__global__ void __launch_bounds__(256, sizeof(T) == 4 ? 2 : 1) k_fused9(const __grid_constant__ KP<T> P, const Fused9P<T> U) {
  typedef P2<T> V;
  typedef typename PairOf<T>::type W2;
  extern __shared__ __align__(16) unsigned char smem9[];
  const int nx = P.nx, nwc = nx >> 6;                 // 64-node column groups (one warp each)
  T* const ring = reinterpret_cast<T*>(smem9);        // [4][nx]
  T* const edge_p = ring + 4 * nx;                    // [4][nwc]: lane 31's +x sends (land in the next group's first column)
  T* const edge_m = edge_p + 4 * nwc;                 // [4][nwc]: lane 0's -x sends (land in the previous group's last column)
  const int lane = threadIdx.x & 31;
  const int c = blockIdx.x;
  const int y0 = (int)((long long)c * P.ny / U.nchunks), y1 = (int)((long long)(c + 1) * P.ny / U.nchunks), rows = y1 - y0;
  for (int i = threadIdx.x; i < 4 * (nx + 2 * nwc); i += blockDim.x) ring[i] = T(0);
  __syncthreads();
  T* const slab = U.part + (long long)c * 2 * nx;
  // flush of the chunk's row k (-1 .. rows), held in ring slot (k + 1) % 4; the slot is left zeroed
  auto flush = [&](int k) {
    const int s = (k + 1) & 3;
    T* const dst = k < 0 ? slab : (k >= rows ? slab + nx : U.phi_dst + (long long)(y0 + k) * nx);
    for (int x0 = 2 * threadIdx.x; x0 < nx; x0 += 2 * blockDim.x) {
      const int wc = x0 >> 6, wl = wc == 0 ? nwc - 1 : wc - 1, wr = wc == nwc - 1 ? 0 : wc + 1;
      W2* p = reinterpret_cast<W2*>(ring + s * nx + x0);
      V v = V(*p);
      *p = V(T(0)).v;
      if (lane == 0) { T& e = edge_p[s * nwc + wl]; v = v + V(e, T(0)); e = T(0); }
      if (lane == 31) { T& e = edge_m[s * nwc + wr]; v = v + V(T(0), e); e = T(0); }
      st_pair<T>(dst + x0, v);
    }
  };
  // one node pair: the step, then where its nine g+ land.  LEAN: no face and no row end next to the pair (warp-uniform choice)
  auto pair = [&](auto lean_tag, const Geo9& geo, int x0, int sm, int sc, int sp) {
    constexpr bool LEAN = decltype(lean_tag)::value;
    V g[Q9];
    step9p_pair<T, LEAN>(P, geo, x0, g);
    V own(T(0));
    Tri9<T> up = {g[dir9(0, 1)], g[dir9(1, 1)], g[dir9(-1, 1)]}, dn = {g[dir9(0, -1)], g[dir9(1, -1)], g[dir9(-1, -1)]};
    Tri9<T> me = {g[0], g[dir9(1, 0)], g[dir9(-1, 0)]};
    if (!LEAN) {
      if (geo.byp) { own = own + ((up.v0 + up.vp) + up.vm); up.v0 = V(T(0)); up.vp = V(T(0)); up.vm = V(T(0)); }
      if (geo.bym) { own = own + ((dn.v0 + dn.vp) + dn.vm); dn.v0 = V(T(0)); dn.vp = V(T(0)); dn.vm = V(T(0)); }
      if (geo.syp) { me.v0 = me.v0 + up.v0; me.vp = me.vp + up.vp; me.vm = me.vm + up.vm; up.v0 = V(T(0)); up.vp = V(T(0)); up.vm = V(T(0)); }
      if (geo.sym) { me.v0 = me.v0 + dn.v0; me.vp = me.vp + dn.vp; me.vm = me.vm + dn.vm; dn.v0 = V(T(0)); dn.vp = V(T(0)); dn.vm = V(T(0)); }
    }
    V cc[3];
    T ep[3], em[3];
    auto finish = [&](Tri9<T> t, V& cv, T& e_p, T& e_m) {
      if (!LEAN) {
        if (geo.bxp) { own = own + V(T(0), t.vp.hi()); t.vp = V(t.vp.lo(), T(0)); }
        if (geo.bxm) { own = own + V(t.vm.lo(), T(0)); t.vm = V(T(0), t.vm.hi()); }
        if (geo.sxp) { t.v0 = t.v0 + V(T(0), t.vp.hi()); t.vp = V(t.vp.lo(), T(0)); }
        if (geo.sxm) { t.v0 = t.v0 + V(t.vm.lo(), T(0)); t.vm = V(T(0), t.vm.hi()); }
      }
      T a = shfl_up1(t.vp.hi()), b = shfl_dn1(t.vm.lo());
      if (lane == 0) a = T(0);
      if (lane == 31) b = T(0);
      cv = (t.v0 + V(a, t.vp.lo())) + V(t.vm.hi(), b);
      e_p = t.vp.hi(); e_m = t.vm.lo();
    };
    finish(up, cc[0], ep[0], em[0]);
    finish(dn, cc[1], ep[1], em[1]);
    finish(me, cc[2], ep[2], em[2]);   // own row last: it also collects what bounced back
    cc[2] = cc[2] + own;
    const int sl[3] = {sp, sm, sc};
    W2* q[3];
    W2 o[3];
#pragma unroll
    for (int k = 0; k < 3; ++k) { q[k] = reinterpret_cast<W2*>(ring + sl[k] * nx + x0); o[k] = *q[k]; }
#pragma unroll
    for (int k = 0; k < 3; ++k) *q[k] = (V(o[k]) + cc[k]).v;
    if (lane == 0 || lane == 31) {
      T* const e = (lane ? edge_p : edge_m) + (x0 >> 6);
#pragma unroll
      for (int k = 0; k < 3; ++k) e[sl[k] * nwc] += lane ? ep[k] : em[k];
    }
  };
#pragma unroll 1
  for (int ly = 0; ly < rows; ++ly) {
    const int y = y0 + ly;
    const int sm = ly & 3, sc = (ly + 1) & 3, sp = (ly + 2) & 3;   // slots of the rows y-1, y, y+1
    const bool yface = (y == 0 && P.bc[2] != BC_PERIODIC) || (y == P.ny - 1 && P.bc[3] != BC_PERIODIC);
    Geo9 lg{};   // the row's part of the lean geometry (rows wrap in y; no face flags)
    {
      const int ym = y > 0 ? y - 1 : P.ny - 1, yp = y < P.ny - 1 ? y + 1 : 0;
      lg.nx = nx;
      lg.r0 = (long long)y * NC9 * nx; lg.rm = (long long)ym * NC9 * nx; lg.rp = (long long)yp * NC9 * nx;
      lg.p0 = y * nx; lg.pm = ym * nx; lg.pp = yp * nx;
    }
#pragma unroll 1
    for (int x0 = 2 * threadIdx.x; x0 < nx; x0 += 2 * blockDim.x) {
      const int wc = x0 >> 6;
      if (yface || wc == 0 || wc == nwc - 1) {
        pair(std::false_type(), make_geo9(P, x0, y), x0, sm, sc, sp);
      } else {
        Geo9 geo = lg;
        geo.x0 = x0;
        pair(std::true_type(), geo, x0, sm, sc, sp);
      }
    }
    __syncthreads();
    flush(ly - 1);
  }
  flush(rows - 1);
  flush(rows);
}

// phi(t+2) of the first and the last row of every chunk: + what the neighbouring chunks sent.  grid = (nchunks, ceil(nx / 4 / 128))
template <typename T> __global__ void __launch_bounds__(128) k_fix9(const __grid_constant__ KP<T> P, const Fused9P<T> U) {
  const int c = blockIdx.x, nx = P.nx;
  const int x0 = 2 * (blockIdx.y * blockDim.x + threadIdx.x);
  if (x0 >= nx) return;
  const int y0 = (int)((long long)c * P.ny / U.nchunks), y1 = (int)((long long)(c + 1) * P.ny / U.nchunks);
  const bool wrap = P.bc[2] == BC_PERIODIC;
  const int cm = c == 0 ? U.nchunks - 1 : c - 1, cp = c == U.nchunks - 1 ? 0 : c + 1;
  if (c > 0 || wrap) {   // the row below sent its +y populations here: halo row 1 (yp) of the chunk below
    T* const r = U.phi_dst + (long long)y0 * nx + x0;
    st_pair<T>(r, ld_pair<T>(r) + ld_pair<T>(U.part + ((long long)cm * 2 + 1) * nx + x0));
  }
  if (c < U.nchunks - 1 || wrap) {
    T* const r = U.phi_dst + (long long)(y1 - 1) * nx + x0;
    st_pair<T>(r, ld_pair<T>(r) + ld_pair<T>(U.part + ((long long)cp * 2) * nx + x0));
  }
}

}  // namespace d2q9
}  // namespace clip
