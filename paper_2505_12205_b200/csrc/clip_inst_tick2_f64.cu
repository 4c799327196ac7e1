// explicit instantiations: k_tick2 launches, double
#include "clip_launch_impl.cuh"
template void clip::launch_tick2<double>(bool, int, unsigned, dim3, cudaStream_t, const clip::FP<double>&, const clip::TickP&, int);
