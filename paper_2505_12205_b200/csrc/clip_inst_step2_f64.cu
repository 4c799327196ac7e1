// explicit instantiations: k_phi2 / k_step2 launches, double
#include "clip_launch_impl.cuh"
template void clip::launch_phi2<double>(int, int, dim3, dim3, cudaStream_t, const clip::FP<double>&);
template void clip::launch_step2<double>(int, bool, int, dim3, dim3, cudaStream_t, const clip::FP<double>&);
