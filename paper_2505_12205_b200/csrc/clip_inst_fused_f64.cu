// explicit instantiations: k_fused / k_fix launches, double
#include "clip_launch_impl.cuh"
template cudaError_t clip::launch_fused<double>(int, int, dim3, dim3, size_t, cudaStream_t, const clip::FP<double>&, const clip::FusedP<double>&);
template void clip::launch_fix<double>(dim3, cudaStream_t, const clip::FP<double>&, const clip::FusedP<double>&);
template cudaError_t clip::launch_fused_tma<double>(int, bool, dim3, dim3, size_t, cudaStream_t, const clip::FP<double>&, const clip::FusedP<double>&);
template cudaError_t clip::launch_fused_cl<double>(int, int, dim3, dim3, size_t, cudaStream_t, const clip::FP<double>&, const clip::FusedP<double>&);
