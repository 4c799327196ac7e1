// clip_launch.cuh -- host-side launch functions of the nx-specialised fast kernels.  They are declared here and DEFINED in
// clip_launch_impl.cuh, which only the small clip_inst_*.cu translation units include (one per kernel family and precision,
// explicit instantiations), so that the ~170 kernel instantiations compile in parallel instead of in one 3-minute unit.
#pragma once
#include "clip_fast.cuh"
#include "clip_fused.cuh"
#include "clip_fused_tma.cuh"

namespace clip {

// Resident threads per SM the k_fused instantiations are compiled for (__launch_bounds__): fp32 384 (<= 168 registers;
// 12 warps with every load of a row in flight beat 16 warps at 128 registers, measured 17.3 vs 16.8 GLUPS at 256^3),
// re-measured in round 2 after the branch-free pull: 17.75 vs 16.81), except 256-thread blocks (nx = 512 and the runtime-nx form),
// which keep 2 blocks, and 96-thread blocks (nx = 192: 5 blocks = 15 warps at 128 registers: the jet lattice); fp64 256 (255 registers).
constexpr int fused_threads_per_sm(int precision, int block_threads) {
  return precision == 32 ? (block_threads >= 256 ? 512 : (block_threads == 96 ? 480 : 384)) : 256;
}


// faces: 0 = all PERIODIC, 1 = the lattice has WALL faces, 2 = it has FREESLIP faces in x / y (and maybe walls); xwalls: non-periodic
// faces in x (k_step2 then keeps 16 warps per SM)
template <typename T> void launch_phi2(int faces, int nx, dim3 g, dim3 b, cudaStream_t st, const FP<T>& F);
template <typename T> void launch_step2(int faces, bool xwalls, int nx, dim3 g, dim3 b, cudaStream_t st, const FP<T>& F);
// returns the CUDA error of the shared-memory opt-in (cudaFuncSetAttribute, once per device and instantiation) or of nothing
template <typename T> cudaError_t launch_fused(int faces, int nx, dim3 g, dim3 b, size_t smem, cudaStream_t st, const FP<T>& F, const FusedP<T>& U);
// cluster form of k_fused (U.cs tiles per thread-block cluster along y; g.x % U.cs == 0)
template <typename T> cudaError_t launch_fused_cl(int faces, int nx, dim3 g, dim3 b, size_t smem, cudaStream_t st, const FP<T>& F, const FusedP<T>& U);
// k_fused_tma (bulk-async feed; periodic x / y faces): same grid and FusedP as k_fused, more shared memory
template <typename T> cudaError_t launch_fused_tma(int nx, bool gonly, dim3 g, dim3 b, size_t smem, cudaStream_t st, const FP<T>& F, const FusedP<T>& U);
template <typename T> void launch_fix(dim3 g, cudaStream_t st, const FP<T>& F, const FusedP<T>& U);

}  // namespace clip
