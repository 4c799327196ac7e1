// clip_static.cu -- clip_outlet_lambda_static (include/clip.h): lambda of the convective outlet (App. B.5, B.22 / B.25,
// PAPER.md:1094-1129) for callers that may not allocate device memory (CUDA graph capture, serving loops, harnesses that forbid
// cudaMalloc).  It is the two-stage computation of the step's k_outlet_lam + k_outlet_reduce (clip_kernels.cuh) with the per-column
// scratch of stage one NOT in a caller workspace but in a file-scope device array of this file; the caller passes only the input
// (u) and the output (lambda).  Nothing here calls cudaMalloc / cudaFree or any allocating routine.
//
// The array `g_scratch` is 2 MiB (CLIP_STATIC_MAX_PLANE_NODES words of 8 bytes): every GPU that loads libclip.so holds it until the
// process exits.  In HOST code the name `g_scratch` is a host-side stand-in, not a device address: the address the kernels get is
// taken once per device with cudaGetSymbolAddress (scratch_of_current_device below).  All calls on one device share the array: calls
// that overlap on the GPU (different streams, no ordering between them) race.  Nothing in it has to start at zero -- stage one
// writes every entry stage two reads, in the same call -- so the contents a previous call left behind are never read.
#include "../../include/clip.h"

#include <cuda_runtime.h>
#include <cstdarg>
#include <cstdint>
#include <cstdio>
#include <mutex>

namespace {

static __device__ __align__(256) unsigned char g_scratch[(size_t)CLIP_STATIC_MAX_PLANE_NODES * 8];

constexpr int MAX_DEVICES = 64;
std::mutex g_mutex;
void* g_scratch_ptr[MAX_DEVICES] = {};   // device address of g_scratch on device d (0: not looked up yet)
thread_local char g_err[256] = "";

int fail(int code, const char* fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(g_err, sizeof g_err, fmt, ap);
  va_end(ap);
  return code;
}

// Device address of g_scratch on the CURRENT device; looked up once per device, with that device current.
int scratch_of_current_device(void** out) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return fail(CLIP_ECUDA, "cudaGetDevice: %s", cudaGetErrorString(e));
  if (dev < 0 || dev >= MAX_DEVICES) return fail(CLIP_EINVAL, "device ordinal %d outside 0 .. %d", dev, MAX_DEVICES - 1);
  std::lock_guard<std::mutex> lock(g_mutex);
  if (!g_scratch_ptr[dev]) {
    void* p = nullptr;
    e = cudaGetSymbolAddress(&p, g_scratch);
    if (e != cudaSuccess || !p) return fail(CLIP_ECUDA, "cudaGetSymbolAddress(g_scratch) on device %d: %s", dev, cudaGetErrorString(e));
    g_scratch_ptr[dev] = p;
  }
  *out = g_scratch_ptr[dev];
  return CLIP_OK;
}

// Stage one (k_outlet_lam with outlet_u_time = 0): U of B.22 per column = u_z of layer N-1 from the stored field u(t)
// (PAPER.md:1107); U_local is clamped here if asked for, the plane-wide schemes in stage two.
template <typename T>
__global__ void __launch_bounds__(256) k_outlet_u_static(const T* __restrict__ uz_layer, long long nxy, int clamp_here, T* __restrict__ scratch) {
  const long long c = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= nxy) return;
  T U = uz_layer[c];
  if (clamp_here && U < T(0)) U = T(0);
  scratch[c] = U;
}

// Stage two (k_outlet_reduce): U_local (mode 0): the column's own value; U_ave (1) / U_max (2): one block, the reduction order of
// k_outlet_reduce (1024 strided partial results, then a tree), so that the result equals the step's bit for bit.
template <typename T>
__global__ void __launch_bounds__(1024) k_outlet_reduce_static(const T* __restrict__ scratch, long long nxy, int mode, int clamp, T* __restrict__ lam) {
  if (mode == 0) {
    for (long long c = threadIdx.x; c < nxy; c += blockDim.x) lam[c] = scratch[c];
    return;
  }
  __shared__ T sh[1024];
  const bool ave = mode == 1;
  T acc = ave ? T(0) : scratch[0];
  for (long long c = threadIdx.x; c < nxy; c += blockDim.x) {
    const T v = scratch[c];
    acc = ave ? acc + v : (v > acc ? v : acc);
  }
  sh[threadIdx.x] = acc;
  __syncthreads();
  for (int s = blockDim.x / 2; s > 0; s >>= 1) {
    if ((int)threadIdx.x < s) {
      const T a = sh[threadIdx.x], b = sh[threadIdx.x + s];
      sh[threadIdx.x] = ave ? a + b : (b > a ? b : a);
    }
    __syncthreads();
  }
  T U = ave ? sh[0] / T(nxy) : sh[0];
  if (clamp && U < T(0)) U = T(0);
  for (long long c = threadIdx.x; c < nxy; c += blockDim.x) lam[c] = U;
}

template <typename T>
int run(const void* d_u, long long nxy, long long n, int nz, int mode, int clamp, void* d_lambda, void* scratch, cudaStream_t s) {
  const T* uz_layer = static_cast<const T*>(d_u) + 2 * n + (long long)(nz - 2) * nxy;
  T* sc = static_cast<T*>(scratch);
  const unsigned blocks = (unsigned)((nxy + 255) / 256);
  k_outlet_u_static<T><<<blocks, 256, 0, s>>>(uz_layer, nxy, mode == 0 && clamp, sc);
  k_outlet_reduce_static<T><<<1, 1024, 0, s>>>(sc, nxy, mode, clamp, static_cast<T*>(d_lambda));
  const cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return fail(CLIP_ECUDA, "clip_outlet_lambda_static launch: %s", cudaGetErrorString(e));
  return CLIP_OK;
}

}  // namespace

extern "C" {

int clip_outlet_lambda_static(const void* d_u, int nx, int ny, int nz, int precision, int outlet_u_mode, int outlet_clamp,
                              void* d_lambda, void* cuda_stream) {
  if (precision != 32 && precision != 64) return fail(CLIP_EINVAL, "precision must be 32 or 64");
  if (nx < 1 || ny < 1 || nz < 2) return fail(CLIP_EINVAL, "nx, ny must be >= 1 and nz >= 2 (the outlet needs layer N-1)");
  const long long nxy = (long long)nx * ny;
  if (nxy > (long long)CLIP_STATIC_MAX_PLANE_NODES)
    return fail(CLIP_EINVAL, "nx * ny = %lld exceeds CLIP_STATIC_MAX_PLANE_NODES = %d, the size of the static scratch array", nxy,
                (int)CLIP_STATIC_MAX_PLANE_NODES);
  if ((double)nxy * nz > 2.0e9) return fail(CLIP_EINVAL, "lattice too large (nx*ny*nz must stay below 2e9)");
  if (outlet_u_mode < 0 || outlet_u_mode > 2) return fail(CLIP_EINVAL, "outlet_u_mode must be 0 (U_local), 1 (U_ave) or 2 (U_max)");
  if (outlet_clamp != 0 && outlet_clamp != 1) return fail(CLIP_EINVAL, "outlet_clamp must be 0 or 1");
  const uintptr_t word = precision == 32 ? 4 : 8;
  if (!d_u || !d_lambda || (uintptr_t)d_u % word || (uintptr_t)d_lambda % word)
    return fail(CLIP_EINVAL, "d_u and d_lambda must be non-NULL device pointers aligned to the word size");
  void* scratch = nullptr;
  const int rc = scratch_of_current_device(&scratch);
  if (rc != CLIP_OK) return rc;
  const long long n = nxy * nz;
  cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
  return precision == 32 ? run<float>(d_u, nxy, n, nz, outlet_u_mode, outlet_clamp, d_lambda, scratch, s)
                         : run<double>(d_u, nxy, n, nz, outlet_u_mode, outlet_clamp, d_lambda, scratch, s);
}

const char* clip_static_last_error(void) { return g_err; }

}  // extern "C"
