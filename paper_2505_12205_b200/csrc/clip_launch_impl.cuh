// clip_launch_impl.cuh -- definitions of the launch functions declared in clip_launch.cuh (see there).
#pragma once
#include "clip_launch.cuh"

// nx values with their own instantiation of the fast kernels (direction offsets as immediates); others take NX = 0.
#ifndef CLIP_NX_LIST
#define CLIP_NX_LIST(X) X(64) X(128) X(192) X(256) X(384) X(512)
#endif

namespace clip {

template <typename T, int W> void launch_phi2_w(int nx, dim3 g, dim3 b, cudaStream_t st, const FP<T>& F) {
  switch (nx) {
#define X(N) case N: k_phi2<T, N, W><<<g, b, 0, st>>>(F); break;
    CLIP_NX_LIST(X)
#undef X
    default: k_phi2<T, 0, W><<<g, b, 0, st>>>(F);
  }
}
template <typename T, int W, int MB> void launch_step2_w(int nx, dim3 g, dim3 b, cudaStream_t st, const FP<T>& F) {
  switch (nx) {
#define X(N) case N: k_step2<T, N, W, MB><<<g, b, 0, st>>>(F); break;
    CLIP_NX_LIST(X)
#undef X
    default: k_step2<T, 0, W, MB><<<g, b, 0, st>>>(F);
  }
}
template <typename T> struct StepMinBlocks { static constexpr int value = 3; };  // k_step2 (128-thread blocks)
template <> struct StepMinBlocks<double> { static constexpr int value = 1; };
template <typename T> struct StepMinBlocksBgk { static constexpr int value = 2; };  // all 19 f stay live: 255 registers
template <> struct StepMinBlocksBgk<double> { static constexpr int value = 1; };
template <typename T> struct StepMinBlocksXWalls { static constexpr int value = 4; };  // 128 registers, 16 warps
template <> struct StepMinBlocksXWalls<double> { static constexpr int value = 1; };

// The opt-in to > 48 KB of dynamic shared memory is a per-DEVICE attribute of the kernel: set it once per device and
// instantiation (a process may drive several GPUs), and report its error.
constexpr int MAX_DEVICES = 64;
template <typename T, int NX, int W> cudaError_t launch_fused_nx(dim3 g, dim3 b, size_t smem, cudaStream_t st, const FP<T>& F, const FusedP<T>& U) {
  constexpr int MAXT = NX ? NX / 2 : 256;
  constexpr int TPSM = fused_threads_per_sm(sizeof(T) == 4 ? 32 : 64, MAXT);
  constexpr int MINB = TPSM / MAXT > 0 ? TPSM / MAXT : 1;
  auto kern = k_fused<T, NX, W, MAXT, MINB>;
  static bool attr_done[MAX_DEVICES] = {};  // per instantiation and device
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 0 || dev >= MAX_DEVICES || !attr_done[dev]) {
    e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024 - 1024);
    if (e != cudaSuccess) return e;
    if (dev >= 0 && dev < MAX_DEVICES) attr_done[dev] = true;
  }
  kern<<<g, b, smem, st>>>(F, U);
  return cudaSuccess;
}
template <typename T, int W> cudaError_t launch_fused_w(int nx, dim3 g, dim3 b, size_t smem, cudaStream_t st, const FP<T>& F, const FusedP<T>& U) {
  switch (nx) {
#define X(N) case N: return launch_fused_nx<T, N, W>(g, b, smem, st, F, U);
    CLIP_NX_LIST(X)
#undef X
    default: return launch_fused_nx<T, 0, W>(g, b, smem, st, F, U);
  }
}


// Lattices with FREESLIP faces in x / y (faces = 2): their own instantiations only for the runtime-nx form and nx = 192 (the
// paper's jet has free-slip side walls); other widths take the runtime-nx kernel.
template <typename T> void launch_phi2(int faces, int nx, dim3 g, dim3 b, cudaStream_t st, const FP<T>& F) {
  if (faces == 2) {
    if (nx == 192) k_phi2<T, 192, 2><<<g, b, 0, st>>>(F);
    else k_phi2<T, 0, 2><<<g, b, 0, st>>>(F);
  } else if (faces) launch_phi2_w<T, 1>(nx, g, b, st, F);
  else launch_phi2_w<T, 0>(nx, g, b, st, F);
}
template <typename T> void launch_step2(int faces, bool xwalls, int nx, dim3 g, dim3 b, cudaStream_t st, const FP<T>& F) {
  if (F.k.collision == 1) {  // BGK: runtime-nx kernels (clip.cu admits it on periodic / walled lattices only)
    if (faces) k_step2_bgk<T, 1, StepMinBlocksBgk<T>::value><<<g, b, 0, st>>>(F);
    else k_step2_bgk<T, 0, StepMinBlocksBgk<T>::value><<<g, b, 0, st>>>(F);
    return;
  }
  // walls in x: most blocks run the wall code, which wants warps more than registers (jet lattice: +6 %)
  if (faces == 2) {
    if (nx == 192) k_step2<T, 192, 2, StepMinBlocksXWalls<T>::value><<<g, b, 0, st>>>(F);
    else k_step2<T, 0, 2, StepMinBlocksXWalls<T>::value><<<g, b, 0, st>>>(F);
  } else if (faces && xwalls) launch_step2_w<T, 1, StepMinBlocksXWalls<T>::value>(nx, g, b, st, F);
  else if (faces) launch_step2_w<T, 1, StepMinBlocks<T>::value>(nx, g, b, st, F);
  else launch_step2_w<T, 0, StepMinBlocks<T>::value>(nx, g, b, st, F);
}
template <typename T> cudaError_t launch_fused(int faces, int nx, dim3 g, dim3 b, size_t smem, cudaStream_t st, const FP<T>& F, const FusedP<T>& U) {
  if (faces == 2) return nx == 192 ? launch_fused_nx<T, 192, 2>(g, b, smem, st, F, U) : launch_fused_nx<T, 0, 2>(g, b, smem, st, F, U);  // as launch_step2
  return faces ? launch_fused_w<T, 1>(nx, g, b, smem, st, F, U) : launch_fused_w<T, 0>(nx, g, b, smem, st, F, U);
}
template <typename T, int NX, int W> cudaError_t launch_fused_cl_nx(dim3 g, dim3 b, size_t smem, cudaStream_t st, const FP<T>& F, const FusedP<T>& U) {
  constexpr int MAXT = NX ? NX / 2 : 256;
  constexpr int TPSM = fused_threads_per_sm(sizeof(T) == 4 ? 32 : 64, MAXT);
  constexpr int MINB = TPSM / MAXT > 0 ? TPSM / MAXT : 1;
  auto kern = k_fused<T, NX, W, MAXT, MINB, true>;
  static bool attr_done[MAX_DEVICES] = {};
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 0 || dev >= MAX_DEVICES || !attr_done[dev]) {
    e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024 - 1024);
    if (e != cudaSuccess) return e;
    if (dev >= 0 && dev < MAX_DEVICES) attr_done[dev] = true;
  }
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = g; cfg.blockDim = b; cfg.dynamicSmemBytes = smem; cfg.stream = st;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeClusterDimension;
  at[0].val.clusterDim.x = (unsigned)U.cs; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
  cfg.attrs = at; cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, kern, F, U);
}
// Cluster form: own instantiations for the widths where clusters are the default (nx = 128, 192); every other width takes the
// runtime-nx kernel (clip_params.cluster_y forced: tests, tuning).
template <typename T> cudaError_t launch_fused_cl(int faces, int nx, dim3 g, dim3 b, size_t smem, cudaStream_t st, const FP<T>& F, const FusedP<T>& U) {
  if (faces == 2) return nx == 192 ? launch_fused_cl_nx<T, 192, 2>(g, b, smem, st, F, U) : launch_fused_cl_nx<T, 0, 2>(g, b, smem, st, F, U);
  if (faces) return nx == 128 ? launch_fused_cl_nx<T, 128, 1>(g, b, smem, st, F, U) : (nx == 192 ? launch_fused_cl_nx<T, 192, 1>(g, b, smem, st, F, U) : launch_fused_cl_nx<T, 0, 1>(g, b, smem, st, F, U));
  return nx == 128 ? launch_fused_cl_nx<T, 128, 0>(g, b, smem, st, F, U) : (nx == 192 ? launch_fused_cl_nx<T, 192, 0>(g, b, smem, st, F, U) : launch_fused_cl_nx<T, 0, 0>(g, b, smem, st, F, U));
}
template <typename T, int NX, bool GONLY> cudaError_t launch_fused_tma_nx(dim3 g, dim3 b, size_t smem, cudaStream_t st, const FP<T>& F, const FusedP<T>& U) {
  constexpr int MAXT = NX ? NX / 2 : 256;
  constexpr int MINB = (GONLY && sizeof(T) == 4 && 384 / MAXT > 0) ? 384 / MAXT : 1;   // hybrid: k_fused's occupancy
  auto kern = k_fused_tma<T, NX, MAXT, MINB, GONLY>;
  static bool attr_done[MAX_DEVICES] = {};
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 0 || dev >= MAX_DEVICES || !attr_done[dev]) {
    e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024 - 1024);
    if (e != cudaSuccess) return e;
    if (dev >= 0 && dev < MAX_DEVICES) attr_done[dev] = true;
  }
  kern<<<g, b, smem, st>>>(F, U);
  return cudaSuccess;
}
template <typename T> cudaError_t launch_fused_tma(int nx, bool gonly, dim3 g, dim3 b, size_t smem, cudaStream_t st, const FP<T>& F, const FusedP<T>& U) {
  if (gonly) {
    switch (nx) {
      case 256: return launch_fused_tma_nx<T, 256, true>(g, b, smem, st, F, U);
      case 512: return launch_fused_tma_nx<T, 512, true>(g, b, smem, st, F, U);
      default: return launch_fused_tma_nx<T, 0, true>(g, b, smem, st, F, U);
    }
  }
  switch (nx) {
    case 128: return launch_fused_tma_nx<T, 128, false>(g, b, smem, st, F, U);
    case 256: return launch_fused_tma_nx<T, 256, false>(g, b, smem, st, F, U);
    case 384: return launch_fused_tma_nx<T, 384, false>(g, b, smem, st, F, U);
    case 512: return launch_fused_tma_nx<T, 512, false>(g, b, smem, st, F, U);
    default: return launch_fused_tma_nx<T, 0, false>(g, b, smem, st, F, U);
  }
}
template <typename T> void launch_fix(dim3 g, cudaStream_t st, const FP<T>& F, const FusedP<T>& U) {
  k_fix<T><<<g, FIX_THREADS, 0, st>>>(F, U);
}

}  // namespace clip
