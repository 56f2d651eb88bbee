// hk_internal.h — helpers shared by the translation units of libhk.so (not part of the C ABI).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/hk.h"

#include <mutex>

namespace hk {

// A step that must run once per DEVICE (cudaFuncSetAttribute, occupancy queries, memory-pool creation): process-wide
// `static bool` latches are wrong for a process that drives several GPUs, and unsynchronised ones race between host threads.
struct PerDeviceOnce {
  std::mutex mu;
  uint64_t done = 0;  // bit d: done on device d (devices >= 64: redone on every call)
  template <class F>
  int run(F &&f)
  {
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return HK_ERR_CUDA;
    std::lock_guard<std::mutex> lk(mu);
    if (dev >= 0 && dev < 64 && ((done >> dev) & 1u)) return HK_OK;
    const int rc = f(dev);
    if (rc == HK_OK && dev >= 0 && dev < 64) done |= (uint64_t)1 << dev;
    return rc;
  }
};

// records the CUDA error text for hk_last_cuda_error() and maps it to HK_ERR_NOMEM / HK_ERR_CUDA
int cuda_fail(cudaError_t e, const char *what);

// Stream-ordered allocations from the library's own memory pool (one per device, created on first use, release
// threshold = unlimited so that scratch freed by one call is reused by the next instead of going back to the driver).
int pool_alloc(void **p, size_t bytes, cudaStream_t st);
void pool_free(void *p, cudaStream_t st);

// hk_sort.cu
int sort_lines_copy(const hk_lines *in, int64_t n, cudaStream_t st, hk_lines *out, void **buf);

// hk_resample.cu: device copy of the projection matrix P[n_c][ppb] of the Chebyshev least-squares fit on the current device
// (factored on the host and uploaded on first use — synchronous — then cached for the life of the process)
int cheb_projection_device(int ppb, int n_c, const double **P_out);

}  // namespace hk
