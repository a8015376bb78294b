// no_alloc.cu - read-back of the HH gates through a staging array that nobody has to allocate.
//
// arb_probe(ARB_PROBE_M / H / N) gathers one gate variable of every HH instance into a per-CV staging buffer on the
// device (zero where a control volume carries no HH mechanism) and copies that buffer to the caller.  Its staging
// buffer is part of the workspace the caller allocates for arb_create.  This file holds the variant for callers that
// may not allocate (code under CUDA graph capture, serving loops, harnesses that forbid cudaMalloc): the staging
// buffer is a file-scope device array of kNoAllocMaxCv doubles, which every GPU that loads the library holds until the
// process exits.
//
//   * In host code the array's NAME is a host-side stand-in, not a device address.  noalloc_scratch() asks the runtime
//     for the address once per device (cudaGetSymbolAddress, with that device current) and the kernels are given that.
//   * All calls on a device share the array, and it keeps what the last call left: every call clears the part it uses
//     before it gathers.  Two calls that overlap on the GPU (different streams, different models) race.
//   * Nothing here calls cudaMalloc, cudaFree or an allocating library routine.
#include <cuda_runtime.h>
#include <stdint.h>

#include <mutex>

#include "kernels.cuh"

namespace arbb {

namespace {

constexpr int kMaxDevices = 64;

static __device__ __align__(256) double g_noalloc_scratch[kNoAllocMaxCv];

std::mutex g_mutex;
double* g_scratch_ptr[kMaxDevices] = {};     // device address of g_noalloc_scratch on device d, once asked for

// The gate gather of kernels.cu (gather_hh_kernel) on the static staging array: first every control volume of the
// model is set to zero, then instance i writes its gate to its control volume.
__global__ void noalloc_clear_kernel(double* scratch, int64_t n_cv) {
  const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i < n_cv) scratch[i] = 0.0;
}
__global__ void noalloc_gather_hh_kernel(const double* state, const uint32_t* m_idx, const uint32_t* stride, const uint32_t* cv,
                                         int which, int64_t n_hh, double* scratch) {
  const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i < n_hh) scratch[cv[i]] = state[m_idx[i] + (uint32_t)which * stride[i]];
}

}  // namespace

int64_t noalloc_max_cv() { return kNoAllocMaxCv; }

// Device address of the static staging array on the CURRENT device (asked for once per device).
cudaError_t noalloc_scratch(double** out) {
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
  std::lock_guard<std::mutex> lock(g_mutex);
  if (!g_scratch_ptr[dev]) {
    double* p = nullptr;
    e = cudaGetSymbolAddress((void**)&p, g_noalloc_scratch);
    if (e != cudaSuccess) return e;
    g_scratch_ptr[dev] = p;
  }
  *out = g_scratch_ptr[dev];
  return cudaSuccess;
}

// Queues on `s`: clear scratch[0, n_cv), gather gate `which` (0 m, 1 h, 2 n) of the n_hh instances into it, copy it to
// host_out.  The caller synchronises the stream.
cudaError_t launch_noalloc_gates(const double* state, const uint32_t* m_idx, const uint32_t* stride, const uint32_t* cv, int which,
                                 int64_t n_hh, int64_t n_cv, double* host_out, cudaStream_t s) {
  if (n_cv <= 0) return cudaSuccess;
  if (n_cv > kNoAllocMaxCv) return cudaErrorInvalidValue;
  double* scratch = nullptr;
  cudaError_t e = noalloc_scratch(&scratch);
  if (e != cudaSuccess) return e;
  noalloc_clear_kernel<<<(unsigned)((n_cv + 255) / 256), 256, 0, s>>>(scratch, n_cv);
  if (n_hh > 0) noalloc_gather_hh_kernel<<<(unsigned)((n_hh + 255) / 256), 256, 0, s>>>(state, m_idx, stride, cv, which, n_hh, scratch);
  e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  return cudaMemcpyAsync(host_out, scratch, 8 * (size_t)n_cv, cudaMemcpyDeviceToHost, s);
}

}  // namespace arbb
