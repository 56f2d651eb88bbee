// hk_resample.cu — SURVEY.md §8(f) rows on top of the k-distribution:
//   f1  Chebyshev resampling of ln kappa(y): the projection matrix P = R^-1 Q^T of the least-squares
//       problem A C = D (A[k][n] = T_n(2 y_k - 1), y_k = (k + 1/2)/ppb, the same for every bin) is factored ONCE on the
//       host by Householder Q-R in long double and kept on the device; the per-bin work — sort, ln, C = P D — runs in
//       kdist_kernel (hk_kdist.cu).  hk_cheb_eval reconstructs kappa(y) = exp(sum_n C_n T_n(2y-1)) by Clenshaw.
//   f2  transmission function (eq. 5; "computing T for 1000 values of m~"):
//       from the k-table, T = sum_q w_q exp(-k_q m~), and directly from kappa(x), T = mean_j exp(-kappa_j m~).
#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>

#include <mutex>
#include <new>
#include <vector>

#include "hk_internal.h"
#include "hk_voigt.cuh"  // exp_fast

namespace hk {

// ---------------------------------------------------------------------------------------------------------
// f1, host part: P[n][k] (n_c x ppb, row-major) with C = P D the least-squares solution of A C = D
// ---------------------------------------------------------------------------------------------------------
static void cheb_projection_host(int ppb, int n_c, std::vector<double> &P)
{
  typedef long double R;
  const int m = ppb, n = n_c;
  std::vector<R> A((size_t)m * n), Q((size_t)m * n, 0.0L), beta(n);  // column-major: X[j*m + i]
  for (int i = 0; i < m; ++i) {
    const R t = 2.0L * (((R)i + 0.5L) / (R)m) - 1.0L;
    A[i] = 1.0L;
    if (n > 1) A[(size_t)m + i] = t;
    for (int j = 2; j < n; ++j) A[(size_t)j * m + i] = 2.0L * t * A[(size_t)(j - 1) * m + i] - A[(size_t)(j - 2) * m + i];
  }
  // Householder: H_j = I - beta_j v_j v_j^T, v_j stored in A[j:, j] (v_j[j] = 1 implied), R in the upper triangle
  std::vector<R> diagR(n);
  for (int j = 0; j < n; ++j) {
    R *a = &A[(size_t)j * m];
    R nrm = 0.0L;
    for (int i = j; i < m; ++i) nrm += a[i] * a[i];
    nrm = sqrtl(nrm);
    const R alpha = a[j] > 0.0L ? -nrm : nrm;
    const R v0 = a[j] - alpha;
    beta[j] = (nrm > 0.0L) ? -v0 / alpha : 0.0L;  // = 2 / (v^T v) with v scaled so that v[j] = 1
    if (v0 != 0.0L)
      for (int i = j + 1; i < m; ++i) a[i] /= v0;
    diagR[j] = alpha;
    for (int c = j + 1; c < n; ++c) {
      R *b = &A[(size_t)c * m];
      R s = b[j];
      for (int i = j + 1; i < m; ++i) s += a[i] * b[i];
      s *= beta[j];
      b[j] -= s;
      for (int i = j + 1; i < m; ++i) b[i] -= s * a[i];
    }
  }
  // thin Q = H_0 H_1 ... H_{n-1} [I_n; 0]
  for (int c = 0; c < n; ++c) Q[(size_t)c * m + c] = 1.0L;
  for (int j = n - 1; j >= 0; --j) {
    const R *v = &A[(size_t)j * m];
    for (int c = 0; c < n; ++c) {
      R *q = &Q[(size_t)c * m];
      R s = q[j];
      for (int i = j + 1; i < m; ++i) s += v[i] * q[i];
      s *= beta[j];
      q[j] -= s;
      for (int i = j + 1; i < m; ++i) q[i] -= s * v[i];
    }
  }
  // P[:, k] = R^-1 (row k of Q)^T by back substitution
  P.assign((size_t)n * m, 0.0);
  std::vector<R> x(n);
  for (int k = 0; k < m; ++k) {
    for (int r = n - 1; r >= 0; --r) {
      R s = Q[(size_t)r * m + k];
      for (int c = r + 1; c < n; ++c) s -= A[(size_t)c * m + r] * x[c];
      x[r] = s / diagR[r];
    }
    for (int r = 0; r < n; ++r) P[(size_t)r * m + k] = (double)x[r];
  }
}

struct ChebEntry {
  int dev, ppb, n_c;
  double *P;
};
static std::mutex g_cheb_mu;
static std::vector<ChebEntry> g_cheb;

// device copy of P for (ppb, n_c) on the current device: built and uploaded on first use (synchronous), then cached
int cheb_projection_device(int ppb, int n_c, const double **P_out)
{
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return cuda_fail(e, "cudaGetDevice");
  std::lock_guard<std::mutex> lk(g_cheb_mu);
  for (const ChebEntry &c : g_cheb)
    if (c.dev == dev && c.ppb == ppb && c.n_c == n_c) {
      *P_out = c.P;
      return HK_OK;
    }
  std::vector<double> P;
  try {
    cheb_projection_host(ppb, n_c, P);
  } catch (const std::bad_alloc &) {
    return HK_ERR_NOMEM;
  }
  double *d = nullptr;
  e = cudaMalloc(&d, P.size() * sizeof(double));
  if (e != cudaSuccess) return cuda_fail(e, "cudaMalloc(cheb P)");
  e = cudaMemcpy(d, P.data(), P.size() * sizeof(double), cudaMemcpyHostToDevice);
  if (e != cudaSuccess) {
    cudaFree(d);
    return cuda_fail(e, "cudaMemcpy(cheb P)");
  }
  g_cheb.push_back({dev, ppb, n_c, d});
  *P_out = d;
  return HK_OK;
}

// ---------------------------------------------------------------------------------------------------------
// kernels
// ---------------------------------------------------------------------------------------------------------
// kappa(y) = exp(sum_n C_n T_n(t)), t = 2y - 1, by the Clenshaw recurrence; one thread per (bin, y)
__global__ void __launch_bounds__(256) cheb_eval_kernel(const double *coef, int64_t n_bins, int n_c, const double *y, int n_y,
                                                        double *out)
{
  const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= n_bins * n_y) return;
  const int64_t b = idx / n_y;
  const double t = fma(2.0, y[idx - b * n_y], -1.0);
  const double *c = coef + b * n_c;
  double b1 = 0.0, b2 = 0.0;
  for (int n = n_c - 1; n >= 1; --n) {
    const double b0 = fma(2.0 * t, b1, c[n] - b2);
    b2 = b1;
    b1 = b0;
  }
  out[idx] = exp(fma(t, b1, c[0] - b2));
}

struct TransArgs {
  const double *k_table;  // [n_bins][n_g]
  const double *mcol;     // [n_m]
  double *T_out;          // [n_bins][n_m]
  int n_g, n_m;
  double w[128];          // Gauss-Legendre weights on (0,1)
};

// T[b][m] = sum_q w_q exp(-k[b][q] m~_m): one CTA per bin, thread per column mass, fixed summation order
__global__ void __launch_bounds__(128) transmission_kernel(const __grid_constant__ TransArgs a)
{
  __shared__ double sk[128];
  const int b = blockIdx.x;
  if (threadIdx.x < a.n_g) sk[threadIdx.x] = a.k_table[(int64_t)b * a.n_g + threadIdx.x];
  __syncthreads();
  for (int m = threadIdx.x; m < a.n_m; m += blockDim.x) {
    const double mm = a.mcol[m];
    double acc = 0.0;
    for (int q = 0; q < a.n_g; ++q) acc = fma(a.w[q], exp_fast(fmax(-sk[q] * mm, -700.0)), acc);  // e^-700: 1e-304
    a.T_out[(int64_t)b * a.n_m + m] = acc;
  }
}

// T[b][m] = (1/ppb) sum_j exp(-kappa_j m~_m) over the bin's points (ascending j: fixed order).  CTA = (bin, 128 column
// masses); the bin's kappa passes through shared memory in chunks and is broadcast to the threads; two independent sums
// (even / odd j) per thread hide the latency of exp.
constexpr int kTdChunk = 2048;
__global__ void __launch_bounds__(128) transmission_direct_kernel(const double *kappa, int ppb, const double *mcol, int n_m,
                                                                 double *T_out)
{
  __shared__ double sk[kTdChunk];
  const int b = blockIdx.x;
  const int m = blockIdx.y * blockDim.x + threadIdx.x;
  const double mm = m < n_m ? -mcol[m] : 0.0;
  const double *src = kappa + (int64_t)b * ppb;
  double s0 = 0.0, s1 = 0.0;
  for (int c0 = 0; c0 < ppb; c0 += kTdChunk) {
    const int cnt = min(kTdChunk, ppb - c0);
    __syncthreads();
    for (int i = threadIdx.x; i < cnt; i += blockDim.x) sk[i] = src[c0 + i];
    __syncthreads();
    int j = 0;
    for (; j + 1 < cnt; j += 2) {
      s0 += exp_fast(fmax(sk[j] * mm, -700.0));  // 16 FP64 instructions, no range guards (e^-700 = 1e-304 stands for 0)
      s1 += exp_fast(fmax(sk[j + 1] * mm, -700.0));
    }
    if (j < cnt) s0 += exp_fast(fmax(sk[j] * mm, -700.0));
  }
  if (m < n_m) T_out[(int64_t)b * n_m + m] = (s0 + s1) / (double)ppb;
}

}  // namespace hk

using namespace hk;

static bool bins_of(int64_t n_points, double dnu, double bin_width, int *ppb_out, int64_t *n_bins_out, int *rc)
{
  *rc = HK_ERR_INVALID;
  if (n_points < 1 || !(dnu > 0.0) || !isfinite(dnu) || !(bin_width > 0.0) || !isfinite(bin_width)) return false;
  const double ratio = bin_width / dnu, ppb_d = nearbyint(ratio);
  if (ppb_d < 1.0 || fabs(ratio - ppb_d) > 1e-9 * ppb_d) return false;
  if (ppb_d > 1.0e9) { *rc = HK_ERR_UNSUPPORTED; return false; }
  const int ppb = (int)ppb_d;
  if (n_points % ppb != 0) return false;
  const int64_t n_bins = n_points / ppb;
  if (n_bins > 2147483647LL) { *rc = HK_ERR_UNSUPPORTED; return false; }
  *ppb_out = ppb;
  *n_bins_out = n_bins;
  *rc = HK_OK;
  return true;
}

extern "C" int hk_cheb_projection(int ppb, int n_c, double *P_host_out)
{
  if (!P_host_out || n_c < 1 || n_c > 64 || ppb < n_c || ppb > 16384) return HK_ERR_INVALID;
  std::vector<double> P;
  try {
    cheb_projection_host(ppb, n_c, P);
  } catch (const std::bad_alloc &) {
    return HK_ERR_NOMEM;
  }
  for (size_t i = 0; i < P.size(); ++i) P_host_out[i] = P[i];
  return HK_OK;
}

extern "C" int hk_cheb_eval(const double *coef, int64_t n_bins, int n_c, const double *y, int n_y, double *kappa_y_out,
                            void *stream)
{
  if (!coef || !y || !kappa_y_out || n_bins < 1 || n_c < 1 || n_c > 64 || n_y < 1) return HK_ERR_INVALID;
  const int64_t total = n_bins * n_y;
  if ((total + 255) / 256 > 2147483647LL) return HK_ERR_UNSUPPORTED;
  cheb_eval_kernel<<<(unsigned)((total + 255) / 256), 256, 0, (cudaStream_t)stream>>>(coef, n_bins, n_c, y, n_y, kappa_y_out);
  cudaError_t e = cudaGetLastError();
  return e == cudaSuccess ? HK_OK : cuda_fail(e, "cheb_eval_kernel launch");
}

extern "C" int hk_transmission(const double *k_table, int64_t n_bins, int n_g, const double *mcol, int n_m, double *T_out,
                               void *stream)
{
  if (!k_table || !mcol || !T_out || n_bins < 1 || n_bins > 2147483647LL || n_g < 1 || n_g > 128 || n_m < 1)
    return HK_ERR_INVALID;
  TransArgs a;
  a.k_table = k_table; a.mcol = mcol; a.T_out = T_out; a.n_g = n_g; a.n_m = n_m;
  double g[128];
  int rc = hk_gauss_legendre(n_g, g, a.w);
  if (rc != HK_OK) return rc;
  transmission_kernel<<<(unsigned)n_bins, 128, 0, (cudaStream_t)stream>>>(a);
  cudaError_t e = cudaGetLastError();
  return e == cudaSuccess ? HK_OK : cuda_fail(e, "transmission_kernel launch");
}

extern "C" int hk_transmission_direct(const double *kappa, int64_t n_points, double dnu, double bin_width, const double *mcol,
                                      int n_m, double *T_out, void *stream)
{
  if (!kappa || !mcol || !T_out || n_m < 1) return HK_ERR_INVALID;
  int ppb = 0, rc = 0;
  int64_t n_bins = 0;
  if (!bins_of(n_points, dnu, bin_width, &ppb, &n_bins, &rc)) return rc;
  const int my = (n_m + 127) / 128;
  if (my > 65535) return HK_ERR_UNSUPPORTED;
  transmission_direct_kernel<<<dim3((unsigned)n_bins, (unsigned)my), 128, 0, (cudaStream_t)stream>>>(kappa, ppb, mcol, n_m, T_out);
  cudaError_t e = cudaGetLastError();
  return e == cudaSuccess ? HK_OK : cuda_fail(e, "transmission_direct_kernel launch");
}
