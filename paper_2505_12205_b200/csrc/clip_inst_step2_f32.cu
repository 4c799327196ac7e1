// explicit instantiations: k_phi2 / k_step2 launches, float
#include "clip_launch_impl.cuh"
template void clip::launch_phi2<float>(int, int, dim3, dim3, cudaStream_t, const clip::FP<float>&);
template void clip::launch_step2<float>(int, bool, int, dim3, dim3, cudaStream_t, const clip::FP<float>&);
