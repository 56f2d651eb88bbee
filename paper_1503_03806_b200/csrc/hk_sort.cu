// hk_sort.cu — orders a copy of an unsorted line list by line centre (prm->lines_sorted == 0).
//
// Not on the timed path: HITRAN / HITEMP files and every BASELINE.json workload arrive wavenumber-ordered, and a
// context (hk_create) sorts once for a whole T-P table.  The key sort itself is the CUDA toolkit's CUB radix sort
// (a library primitive, like calling cuBLAS for a plain GEMM); the gather of the record fields is ours.
#include <cub/device/device_radix_sort.cuh>
#include <cuda_runtime.h>
#include <stdint.h>

#include "hk_internal.h"

namespace hk {

__global__ void __launch_bounds__(256) iota_kernel(int *idx, int64_t n)
{
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) idx[i] = (int)i;
}

// dst_f[i] = src_f[perm[i]] for up to four optional fields (a NULL source leaves its destination untouched)
__global__ void __launch_bounds__(256) gather_fields_kernel(const int *perm, int64_t n, const double *s0, const double *s1,
                                                            const double *s2, const double *s3, double *d0, double *d1,
                                                            double *d2, double *d3)
{
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const int p = perm[i];
  if (s0) d0[i] = s0[p];
  if (s1) d1[i] = s1[p];
  if (s2) d2[i] = s2[p];
  if (s3) d3[i] = s3[p];
}

// Stable ascending sort by nu0.  `buf` receives one allocation holding the ordered copies (freed by the caller with
// pool_free); `out` points into it (optional fields stay NULL when the input has none).
int sort_lines_copy(const hk_lines *in, int64_t n, cudaStream_t st, hk_lines *out, void **buf)
{
  *buf = nullptr;
  const int nf = 3 + (in->n_T ? 1 : 0) + (in->E_low ? 1 : 0) + (in->gamma_self ? 1 : 0) + (in->A21 ? 1 : 0) + (in->delta ? 1 : 0);
  const size_t fbytes = ((size_t)n * sizeof(double) + 255) & ~(size_t)255;
  const size_t ibytes = ((size_t)n * sizeof(int) + 255) & ~(size_t)255;
  size_t tmp_bytes = 0;
  cudaError_t e = cub::DeviceRadixSort::SortPairs(nullptr, tmp_bytes, (const double *)nullptr, (double *)nullptr,
                                                  (const int *)nullptr, (int *)nullptr, (int)n, 0, 64, st);
  if (e != cudaSuccess) return cuda_fail(e, "cub::DeviceRadixSort (size query)");
  void *keep = nullptr, *scratch = nullptr;
  int rc = pool_alloc(&keep, fbytes * nf, st);
  if (rc != HK_OK) return rc;
  rc = pool_alloc(&scratch, 2 * ibytes + tmp_bytes, st);
  if (rc != HK_OK) {
    pool_free(keep, st);
    return rc;
  }
  double *f = (double *)keep;
  int *idx_in = (int *)scratch, *idx_out = (int *)((char *)scratch + ibytes);
  void *tmp = (char *)scratch + 2 * ibytes;
  const unsigned blocks = (unsigned)((n + 255) / 256);
  iota_kernel<<<blocks, 256, 0, st>>>(idx_in, n);
  e = cub::DeviceRadixSort::SortPairs(tmp, tmp_bytes, in->nu0, f, idx_in, idx_out, (int)n, 0, 64, st);
  if (e == cudaSuccess) {
    double *dS = (double *)((char *)keep + fbytes), *dG = (double *)((char *)keep + 2 * fbytes);
    double *dN = in->n_T ? (double *)((char *)keep + 3 * fbytes) : nullptr;
    double *dE = in->E_low ? (double *)((char *)keep + (size_t)(3 + (in->n_T ? 1 : 0)) * fbytes) : nullptr;
    int used = 3 + (in->n_T ? 1 : 0) + (in->E_low ? 1 : 0);
    double *dGs = in->gamma_self ? (double *)((char *)keep + (size_t)(used++) * fbytes) : nullptr;
    double *dA = in->A21 ? (double *)((char *)keep + (size_t)(used++) * fbytes) : nullptr;
    double *dD = in->delta ? (double *)((char *)keep + (size_t)(used++) * fbytes) : nullptr;
    gather_fields_kernel<<<blocks, 256, 0, st>>>(idx_out, n, in->S, in->gamma0, in->n_T, in->E_low, dS, dG, dN, dE);
    if (dGs || dA || dD)
      gather_fields_kernel<<<blocks, 256, 0, st>>>(idx_out, n, in->gamma_self, in->A21, in->delta, nullptr, dGs, dA, dD,
                                                   nullptr);
    e = cudaGetLastError();
    out->gamma_self = dGs;
    out->A21 = dA;
    out->delta = dD;  // eq. 21 is applied by a1: the list is ordered by the unshifted centres
    out->nu0 = f;
    out->S = dS;
    out->gamma0 = dG;
    out->n_T = dN;
    out->E_low = dE;
  }
  pool_free(scratch, st);
  if (e != cudaSuccess) {
    pool_free(keep, st);
    return cuda_fail(e, "sort_lines_copy");
  }
  *buf = keep;
  return HK_OK;
}

}  // namespace hk
