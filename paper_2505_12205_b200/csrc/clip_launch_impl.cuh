// clip_launch_impl.cuh -- definitions of the launch functions declared in clip_launch.cuh (see there).
#pragma once
#include "clip_launch.cuh"

// nx values with their own instantiation of the fast kernels (direction offsets as immediates); others take NX = 0.
#ifndef CLIP_NX_LIST
#define CLIP_NX_LIST(X) X(64) X(128) X(192) X(256) X(384) X(512)
#endif

namespace clip {

template <typename T, bool W> void launch_phi2_w(int nx, dim3 g, dim3 b, cudaStream_t st, const FP<T>& F) {
  switch (nx) {
#define X(N) case N: k_phi2<T, N, W><<<g, b, 0, st>>>(F); break;
    CLIP_NX_LIST(X)
#undef X
    default: k_phi2<T, 0, W><<<g, b, 0, st>>>(F);
  }
}
template <typename T, bool W, int MB> void launch_step2_w(int nx, dim3 g, dim3 b, cudaStream_t st, const FP<T>& F) {
  switch (nx) {
#define X(N) case N: k_step2<T, N, W, MB><<<g, b, 0, st>>>(F); break;
    CLIP_NX_LIST(X)
#undef X
    default: k_step2<T, 0, W, MB><<<g, b, 0, st>>>(F);
  }
}
template <typename T, bool W, int MB>
void launch_tick2_w(int nx, unsigned items, dim3 b, cudaStream_t st, const FP<T>& F, const TickP& tk, int lag) {
  switch (nx) {
#define X(N) case N: k_tick2<T, N, W, MB><<<items, b, 0, st>>>(F, tk, lag); break;
    CLIP_NX_LIST(X)
#undef X
    default: k_tick2<T, 0, W, MB><<<items, b, 0, st>>>(F, tk, lag);
  }
}
template <typename T> struct StepMinBlocks { static constexpr int value = 3; };  // k_step2 (128-thread blocks)
template <> struct StepMinBlocks<double> { static constexpr int value = 1; };
template <typename T> struct StepMinBlocksXWalls { static constexpr int value = 4; };  // 128 registers, 16 warps
template <> struct StepMinBlocksXWalls<double> { static constexpr int value = 1; };
template <typename T> struct TickMinBlocks { static constexpr int value = 2; };  // k_tick2 (__launch_bounds__(256, .))
template <> struct TickMinBlocks<double> { static constexpr int value = 1; };

template <typename T, int NX, bool W> void launch_fused_nx(dim3 g, dim3 b, size_t smem, cudaStream_t st, const FP<T>& F, const FusedP<T>& U) {
  constexpr int MAXT = NX ? NX / 2 : 256;
  constexpr int TPSM = fused_threads_per_sm(sizeof(T) == 4 ? 32 : 64, MAXT);
  constexpr int MINB = TPSM / MAXT > 0 ? TPSM / MAXT : 1;
  auto kern = k_fused<T, NX, W, MAXT, MINB>;
  static bool attr_done = false;  // per instantiation
  if (!attr_done) { cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024 - 1024); attr_done = true; }
  kern<<<g, b, smem, st>>>(F, U);
}
template <typename T, bool W> void launch_fused_w(int nx, dim3 g, dim3 b, size_t smem, cudaStream_t st, const FP<T>& F, const FusedP<T>& U) {
  switch (nx) {
#define X(N) case N: launch_fused_nx<T, N, W>(g, b, smem, st, F, U); break;
    CLIP_NX_LIST(X)
#undef X
    default: launch_fused_nx<T, 0, W>(g, b, smem, st, F, U);
  }
}


template <typename T> void launch_phi2(bool walls, int nx, dim3 g, dim3 b, cudaStream_t st, const FP<T>& F) {
  if (walls) launch_phi2_w<T, true>(nx, g, b, st, F);
  else launch_phi2_w<T, false>(nx, g, b, st, F);
}
template <typename T> void launch_step2(bool walls, bool xwalls, int nx, dim3 g, dim3 b, cudaStream_t st, const FP<T>& F) {
  // walls in x: most blocks run the branchy wall code, which wants warps more than registers (jet lattice: +6 %)
  if (walls && xwalls) launch_step2_w<T, true, StepMinBlocksXWalls<T>::value>(nx, g, b, st, F);
  else if (walls) launch_step2_w<T, true, StepMinBlocks<T>::value>(nx, g, b, st, F);
  else launch_step2_w<T, false, StepMinBlocks<T>::value>(nx, g, b, st, F);
}
template <typename T> void launch_tick2(bool walls, int nx, unsigned items, dim3 b, cudaStream_t st, const FP<T>& F, const TickP& tk, int lag) {
  if (walls) launch_tick2_w<T, true, TickMinBlocks<T>::value>(nx, items, b, st, F, tk, lag);
  else launch_tick2_w<T, false, TickMinBlocks<T>::value>(nx, items, b, st, F, tk, lag);
}
template <typename T> void launch_fused(bool walls, int nx, dim3 g, dim3 b, size_t smem, cudaStream_t st, const FP<T>& F, const FusedP<T>& U) {
  if (walls) launch_fused_w<T, true>(nx, g, b, smem, st, F, U);
  else launch_fused_w<T, false>(nx, g, b, smem, st, F, U);
}
template <typename T> void launch_fix(dim3 g, cudaStream_t st, const FP<T>& F, const FusedP<T>& U) {
  k_fix<T><<<g, FIX_THREADS, 0, st>>>(F, U);
}

}  // namespace clip
