// clip_pack.cuh -- two-lane packed arithmetic for the fast kernels: one thread owns two x-adjacent lattice nodes.
//
// fp32: the pair lives in a 64-bit register pair and every operation is one packed Blackwell instruction
// (FADD2 / FMUL2 / FFMA2, sm_100a), i.e. half the issue slots of scalar code -- the fused step is issue-bound in
// scalar form (profiles/r01_d0_256_fp32.md: 1476 thread instructions per node).  fp64: two plain doubles (DFMA has
// no packed form); the source is shared.
#pragma once
#include <cuda_runtime.h>

namespace clip {

template <typename T> struct P2;  // packed pair of T

template <> struct P2<float> {
  float2 v;
  __device__ __forceinline__ P2() {}
  __device__ __forceinline__ P2(float s) : v(make_float2(s, s)) {}
  __device__ __forceinline__ P2(float a, float b) : v(make_float2(a, b)) {}
  __device__ __forceinline__ explicit P2(float2 a) : v(a) {}
  __device__ __forceinline__ float lo() const { return v.x; }
  __device__ __forceinline__ float hi() const { return v.y; }
};
template <> struct P2<double> {
  double2 v;
  __device__ __forceinline__ P2() {}
  __device__ __forceinline__ P2(double s) : v(make_double2(s, s)) {}
  __device__ __forceinline__ P2(double a, double b) : v(make_double2(a, b)) {}
  __device__ __forceinline__ explicit P2(double2 a) : v(a) {}
  __device__ __forceinline__ double lo() const { return v.x; }
  __device__ __forceinline__ double hi() const { return v.y; }
};

// ---- fp32: packed instructions
__device__ __forceinline__ P2<float> operator+(P2<float> a, P2<float> b) { return P2<float>(__fadd2_rn(a.v, b.v)); }
__device__ __forceinline__ P2<float> operator*(P2<float> a, P2<float> b) { return P2<float>(__fmul2_rn(a.v, b.v)); }
__device__ __forceinline__ P2<float> operator-(P2<float> a) { return P2<float>(-a.v.x, -a.v.y); }
__device__ __forceinline__ P2<float> operator-(P2<float> a, P2<float> b) {
  return P2<float>(__ffma2_rn(b.v, make_float2(-1.f, -1.f), a.v));  // a - b, exact (one rounding)
}
__device__ __forceinline__ P2<float> fma2(P2<float> a, P2<float> b, P2<float> c) { return P2<float>(__ffma2_rn(a.v, b.v, c.v)); }
// a*b - c
__device__ __forceinline__ P2<float> fms2(P2<float> a, P2<float> b, P2<float> c) { return fma2(a, b, -c); }

// ---- fp64: two scalars
__device__ __forceinline__ P2<double> operator+(P2<double> a, P2<double> b) { return P2<double>(a.v.x + b.v.x, a.v.y + b.v.y); }
__device__ __forceinline__ P2<double> operator*(P2<double> a, P2<double> b) { return P2<double>(a.v.x * b.v.x, a.v.y * b.v.y); }
__device__ __forceinline__ P2<double> operator-(P2<double> a) { return P2<double>(-a.v.x, -a.v.y); }
__device__ __forceinline__ P2<double> operator-(P2<double> a, P2<double> b) { return P2<double>(a.v.x - b.v.x, a.v.y - b.v.y); }
__device__ __forceinline__ P2<double> fma2(P2<double> a, P2<double> b, P2<double> c) {
  return P2<double>(fma(a.v.x, b.v.x, c.v.x), fma(a.v.y, b.v.y, c.v.y));
}
__device__ __forceinline__ P2<double> fms2(P2<double> a, P2<double> b, P2<double> c) { return fma2(a, b, -c); }

// ---- per-lane IEEE division / square root (no packed form exists)
__device__ __forceinline__ P2<float> rcp2(P2<float> a) { return P2<float>(1.0f / a.v.x, 1.0f / a.v.y); }
__device__ __forceinline__ P2<double> rcp2(P2<double> a) { return P2<double>(1.0 / a.v.x, 1.0 / a.v.y); }
__device__ __forceinline__ P2<float> sqrt2(P2<float> a) { return P2<float>(sqrtf(a.v.x), sqrtf(a.v.y)); }
__device__ __forceinline__ P2<double> sqrt2(P2<double> a) { return P2<double>(sqrt(a.v.x), sqrt(a.v.y)); }

// ---- global memory: aligned pair access (8 B for float, 16 B for double) and scalar lanes, with a cache hint H:
//   LD_NC  read-only path (ld.global.nc), default          ST_WB  plain store
//   LD_CS  streaming, evict-first in L1/L2 (last use)      ST_CS  streaming store
//   LD_CA  coherent load cached in L1 (data written earlier in the same launch by other blocks)
enum { LD_NC = 0, LD_CS = 1, LD_CA = 2 };
enum { ST_WB = 0, ST_CS = 1 };
template <int H, typename U> __device__ __forceinline__ U ld_hint(const U* p) {
  if (H == LD_CS) return __ldcs(p);
  if (H == LD_CA) return __ldca(p);
  return __ldg(p);
}
template <typename T> struct PairOf;
template <> struct PairOf<float> { typedef float2 type; };
template <> struct PairOf<double> { typedef double2 type; };
template <typename T, int H = LD_NC> __device__ __forceinline__ P2<T> ld_pair(const T* __restrict__ p) {
  return P2<T>(ld_hint<H>(reinterpret_cast<const typename PairOf<T>::type*>(p)));
}
template <typename T, int H = LD_NC> __device__ __forceinline__ T ld_one(const T* __restrict__ p) { return ld_hint<H>(p); }
template <typename T, int H = ST_WB> __device__ __forceinline__ void st_pair(T* __restrict__ p, P2<T> v) {
  typedef typename PairOf<T>::type U;
  if (H == ST_CS) __stcs(reinterpret_cast<U*>(p), v.v);
  else *reinterpret_cast<U*>(p) = v.v;
}

}  // namespace clip
