// explicit instantiations: k_fused / k_fix launches, float
#include "clip_launch_impl.cuh"
template cudaError_t clip::launch_fused<float>(int, int, dim3, dim3, size_t, cudaStream_t, const clip::FP<float>&, const clip::FusedP<float>&);
template void clip::launch_fix<float>(dim3, cudaStream_t, const clip::FP<float>&, const clip::FusedP<float>&);
template cudaError_t clip::launch_fused_tma<float>(int, bool, dim3, dim3, size_t, cudaStream_t, const clip::FP<float>&, const clip::FusedP<float>&);
template cudaError_t clip::launch_fused_cl<float>(int, int, dim3, dim3, size_t, cudaStream_t, const clip::FP<float>&, const clip::FusedP<float>&);
