// explicit instantiations: k_tick2 launches, float
#include "clip_launch_impl.cuh"
template void clip::launch_tick2<float>(bool, int, unsigned, dim3, cudaStream_t, const clip::FP<float>&, const clip::TickP&, int);
