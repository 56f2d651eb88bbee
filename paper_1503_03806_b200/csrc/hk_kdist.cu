// hk_kdist.cu — a5 + a6: per-bin ascending sort of kappa and resampling at Gauss-Legendre nodes (the k-distribution;
// eqs. 14-15, per-bin result PAPER.md:219; the paper sorts the whole grid with Thrust and a bin key).
//
// One CTA per bin.  The bin is padded with +inf to n = T*E points (a power of two) and sorted by a bitonic network held in
// REGISTERS: thread t owns the E consecutive elements t*E .. t*E+E-1.  Every merge phase (block size k) is the "flip"
// step (partner i ^ (k-1)) followed by half-cleaners (partner i ^ j, j = k/4 .. 1), all ascending, so no direction flags:
//   partner in the same thread (j < E)            -> compile-time register pairs
//   partner in the same warp   (j < 32 E)         -> SHFL.BFLY
//   partner in another warp    (j >= 32 E)        -> through shared memory (n = 1024, E = 8: 3 of the 55 steps)
// kappa >= 0 (or +inf), no NaN: plain FP64 compares order the values.  HBM-bound in principle (8 B/point read once,
// 8 n_g B/bin written); in practice bound by the compare-exchange count, n log^2 n / 4 per bin.
#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>

#include "hk_internal.h"

namespace hk {

constexpr unsigned kFullMask = 0xffffffffu;

struct KdistArgs {
  const double *kappa;
  double *k_out;
  int ppb;   // points per bin
  int n;     // padded size, T*E
  int n_g;
  double *ln_out;  // f1 (hk_kdist_cheb): ln max(s_k, 1e-300) of every sorted bin, [n_bins][ppb] scratch, or NULL
  double g[128];
};

// a > b for kappa >= 0 or +inf (no NaN, no -0): the order of the values is the order of their bit patterns as integers
__device__ __forceinline__ bool gt(double a, double b)
{
#ifdef HK_KDIST_INTCMP
  return __double_as_longlong(a) > __double_as_longlong(b);
#else
  return a > b;
#endif
}

__device__ __forceinline__ void ce(double &a, double &b)  // ascending compare-exchange
{
  const bool sw = gt(a, b);
  const double lo = sw ? b : a, hi = sw ? a : b;
  a = lo;
  b = hi;
}

// in-thread half-cleaners j = J, J/2, ..., 1 on E registers
template <int E, int J>
__device__ __forceinline__ void clean_regs(double (&v)[E])
{
  if constexpr (J >= 1) {
#pragma unroll
    for (int r = 0; r < E; ++r)
      if ((r & J) == 0) ce(v[r], v[r | J]);
    clean_regs<E, J / 2>(v);
  }
}
// in-thread flip of block size K <= E
template <int E, int K>
__device__ __forceinline__ void flip_regs(double (&v)[E])
{
#pragma unroll
  for (int r = 0; r < E; ++r)
    if ((r & (K / 2)) == 0) ce(v[r], v[r ^ (K - 1)]);
}
// sorts the E registers of one thread (phases k = 2 .. E)
template <int E, int K>
__device__ __forceinline__ void sort_regs(double (&v)[E])
{
  if constexpr (K <= E) {
    flip_regs<E, K>(v);
    clean_regs<E, K / 4>(v);
    sort_regs<E, K * 2>(v);
  }
}

// shared-memory index of element i: E doubles of a thread, then 2 doubles of padding (128-bit accesses of the blocked
// layout are then conflict-free per quarter warp)
template <int E>
__device__ __forceinline__ int pad(int i)
{
  return i + 2 * (i / E);
}

template <int E, int MAXT, bool CHEB>
__global__ void __launch_bounds__(MAXT) kdist_kernel(const __grid_constant__ KdistArgs a)
{
  extern __shared__ __align__(16) double s[];
  const int T = blockDim.x, t = threadIdx.x;
  const int bin = blockIdx.x;
  const double *src = a.kappa + (int64_t)bin * a.ppb;
  const double inf = __longlong_as_double(0x7ff0000000000000LL);

  double v[E];
  const int i0 = t * E;
  if (i0 + E <= a.ppb && (reinterpret_cast<uintptr_t>(src + i0) & 15) == 0) {
#pragma unroll
    for (int r = 0; r < E; r += 2) {
      const double2 d = *reinterpret_cast<const double2 *>(src + i0 + r);
      v[r] = d.x;
      v[r + 1] = d.y;
    }
  } else {
#pragma unroll
    for (int r = 0; r < E; ++r) v[r] = (i0 + r < a.ppb) ? src[i0 + r] : inf;
  }

  sort_regs<E, 2>(v);

  for (int m = 2; m <= T; m <<= 1) {  // merge phase of block size k = m*E elements = m threads
    // ---- steps whose partner sits in another warp: through shared memory ----
    if (m > 32) {
      __syncthreads();  // previous readers of s are done
#pragma unroll
      for (int r = 0; r < E; r += 2) *reinterpret_cast<double2 *>(&s[pad<E>(i0 + r)]) = make_double2(v[r], v[r + 1]);
      __syncthreads();
      const int k = m * E;
      for (int q = 0; q < E / 2; ++q) {  // flip: i in the lower half of its block, partner i ^ (k-1)
        const int p = t + T * q;
        const int i = ((p & ~(k / 2 - 1)) << 1) | (p & (k / 2 - 1));
        const int x = pad<E>(i), y = pad<E>(i ^ (k - 1));
        const double u = s[x], w = s[y];
        if (gt(u, w)) { s[x] = w; s[y] = u; }
      }
      __syncthreads();
      for (int jj = m >> 2; jj >= 32; jj >>= 1) {
        const int j = jj * E;
        for (int q = 0; q < E / 2; ++q) {
          const int p = t + T * q;
          const int i = ((p & ~(j - 1)) << 1) | (p & (j - 1));
          const int x = pad<E>(i), y = pad<E>(i | j);
          const double u = s[x], w = s[y];
          if (gt(u, w)) { s[x] = w; s[y] = u; }
        }
        __syncthreads();
      }
#pragma unroll
      for (int r = 0; r < E; r += 2) {
        const double2 d = *reinterpret_cast<const double2 *>(&s[pad<E>(i0 + r)]);
        v[r] = d.x;
        v[r + 1] = d.y;
      }
    } else {
      // flip inside the warp: partner thread t ^ (m-1), its register E-1-r; the lower thread keeps the minimum
      const bool keep_min = (t & (m >> 1)) == 0;
#pragma unroll
      for (int r = 0; r < E / 2; ++r) {
        const double oa = __shfl_xor_sync(kFullMask, v[E - 1 - r], m - 1);
        const double ob = __shfl_xor_sync(kFullMask, v[r], m - 1);
        v[r] = (gt(v[r], oa) == keep_min) ? oa : v[r];
        v[E - 1 - r] = (gt(v[E - 1 - r], ob) == keep_min) ? ob : v[E - 1 - r];
      }
    }
    // ---- half-cleaners inside the warp ----
    for (int jj = min(m >> 2, 16); jj >= 1; jj >>= 1) {
      const bool keep_min = (t & jj) == 0;
#pragma unroll
      for (int r = 0; r < E; ++r) {
        const double o = __shfl_xor_sync(kFullMask, v[r], jj);
        const bool take = gt(v[r], o) == keep_min;
        v[r] = take ? o : v[r];
      }
    }
    // ---- half-cleaners inside the thread ----
    clean_regs<E, E / 2>(v);
  }

  // ---- a6: y_k = (k + 1/2)/ppb, linear interpolation at the Gauss-Legendre nodes, clamped at the ends ----
  __syncthreads();
#pragma unroll
  for (int r = 0; r < E; r += 2) *reinterpret_cast<double2 *>(&s[pad<E>(i0 + r)]) = make_double2(v[r], v[r + 1]);
  __syncthreads();
  for (int q = t; a.k_out && q < a.n_g; q += T) {
    const double p = __dadd_rn(__dmul_rn(a.g[q], (double)a.ppb), -0.5);
    double val;
    if (p <= 0.0) val = s[pad<E>(0)];
    else if (p >= (double)(a.ppb - 1)) val = s[pad<E>(a.ppb - 1)];
    else {
      const int k = (int)floor(p);
      const double f = p - (double)k;
      const double s0 = s[pad<E>(k)], s1 = s[pad<E>(k + 1)];
      val = s0 + f * (s1 - s0);
    }
    a.k_out[(int64_t)bin * a.n_g + q] = val;
  }
  // ---- f1: D_k = ln max(s_k, 1e-300) of the sorted bin, for the Chebyshev least-squares fit (cheb_project_kernel)
  if constexpr (CHEB) {
    double *dst = a.ln_out + (int64_t)bin * a.ppb;
#pragma unroll
    for (int r = 0; r < E; ++r)
      if (i0 + r < a.ppb) dst[i0 + r] = log(fmax(v[r], 1.0e-300));
  }
}

// f1: C = D P^T, the Chebyshev coefficients of ln kappa(y) of every bin (the Q-R factorisation behind
// P is done once on the host, hk_resample.cu).  D [n_bins][ppb] (written by kdist_kernel), P [n_c][ppb], C [n_bins][n_c].
// A plain FP64 contraction of 2 n_bins ppb n_c flop (1.2e8 at config 1: microseconds of the FP64 pipe, so no tensor-core
// path); what matters is that P is read once per 8 bins, not once per bin, and that enough CTAs are in flight to hide the
// staging: CTA = 8 bins x all coefficients, D and P staged through (dynamic) shared memory in chunks of up to 256 points
// (few, long stages: every load of a stage is in flight at once); thread t owns bin t % 8 and the coefficients t / 8,
// t / 8 + 16, ...; fixed summation order.
constexpr int kCpBins = 8, kCpChunk = 256, kCpMaxNc = 64, kCpGroups = 128 / kCpBins;
__global__ void __launch_bounds__(128) cheb_project_kernel(const double *D, const double *P, int64_t n_bins, int ppb, int n_c,
                                                           double *C)
{
  extern __shared__ __align__(16) double cp_smem[];
  const int KC = min(kCpChunk, ppb), ld = KC + 1;
  double *Ds = cp_smem;               // [kCpBins][ld]
  double *Ps = cp_smem + kCpBins * ld;  // [n_c][ld]
  const int t = threadIdx.x, bl = t % kCpBins, cg = t / kCpBins;
  const int64_t b0 = (int64_t)blockIdx.x * kCpBins;
  const int nb = (int)min((int64_t)kCpBins, n_bins - b0);
  constexpr int U = kCpMaxNc / kCpGroups;
  double acc[U];
#pragma unroll
  for (int u = 0; u < U; ++u) acc[u] = 0.0;
  for (int k0 = 0; k0 < ppb; k0 += KC) {
    const int kc = min(KC, ppb - k0);
    __syncthreads();
    // thread t stages columns t and t + 128 of every row; loads go to registers in batches of 8 rows before any store, so
    // that a batch is one round trip to L2.  Every CTA stages the same rows of P at about the same time: each starts at
    // another row, so that their requests spread over the L2 slices instead of queueing on one line.
    constexpr int H = kCpChunk / 128;
    {
      double tmp[kCpBins][H];
#pragma unroll
      for (int r = 0; r < kCpBins; ++r)
#pragma unroll
        for (int h = 0; h < H; ++h) {
          const int c = t + 128 * h;
          tmp[r][h] = (r < nb && c < kc) ? D[(b0 + r) * ppb + k0 + c] : 0.0;
        }
#pragma unroll
      for (int r = 0; r < kCpBins; ++r)
#pragma unroll
        for (int h = 0; h < H; ++h)
          if (t + 128 * h < KC) Ds[r * ld + t + 128 * h] = tmp[r][h];
    }
    const int r_first = (int)(blockIdx.x % (unsigned)n_c);
    for (int r0 = 0; r0 < n_c; r0 += 8) {
      double tmp[8][H];
      int row[8];
#pragma unroll
      for (int q = 0; q < 8; ++q) {
        const int rr = min(r0 + q, n_c - 1) + r_first;
        row[q] = rr < n_c ? rr : rr - n_c;
#pragma unroll
        for (int h = 0; h < H; ++h) {
          const int c = t + 128 * h;
          tmp[q][h] = c < kc ? __ldg(P + (int64_t)row[q] * ppb + k0 + c) : 0.0;
        }
      }
#pragma unroll
      for (int q = 0; q < 8; ++q)
#pragma unroll
        for (int h = 0; h < H; ++h)
          if (r0 + q < n_c && t + 128 * h < KC) Ps[row[q] * ld + t + 128 * h] = tmp[q][h];
    }
    __syncthreads();
#pragma unroll 8
    for (int kk = 0; kk < kc; ++kk) {
      const double dv = Ds[bl * ld + kk];
#pragma unroll
      for (int u = 0; u < U; ++u)
        if (cg + kCpGroups * u < n_c) acc[u] = fma(Ps[(cg + kCpGroups * u) * ld + kk], dv, acc[u]);
    }
  }
  if (bl < nb) {
#pragma unroll
    for (int u = 0; u < U; ++u)
      if (cg + kCpGroups * u < n_c) C[(b0 + bl) * n_c + cg + kCpGroups * u] = acc[u];
  }
}

template <int E, int MAXT, bool CHEB>
static int launch_kdist_t(const KdistArgs &a, int64_t n_bins, cudaStream_t st)
{
  const int T = a.n / E;
  const size_t smem = (size_t)(a.n + 2 * T) * sizeof(double);
  static PerDeviceOnce attr;  // one per instantiation; the attribute is a per-device setting
  const int rca = attr.run([](int) {
    cudaError_t e = cudaFuncSetAttribute(kdist_kernel<E, MAXT, CHEB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (16384 + 2048) * 8);
    return e == cudaSuccess ? HK_OK : cuda_fail(e, "cudaFuncSetAttribute(kdist_kernel)");
  });
  if (rca != HK_OK) return rca;
  kdist_kernel<E, MAXT, CHEB><<<(unsigned)n_bins, T, smem, st>>>(a);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return cuda_fail(e, "kdist_kernel launch");
  return HK_OK;
}

// the plain k-distribution (a5 + a6) and the variant with the Chebyshev epilogue are separate instantiations: the epilogue's
// registers do not weigh on the hot path
template <int E, int MAXT>
static int launch_kdist(const KdistArgs &a, int64_t n_bins, cudaStream_t st)
{
  return a.ln_out ? launch_kdist_t<E, MAXT, true>(a, n_bins, st) : launch_kdist_t<E, MAXT, false>(a, n_bins, st);
}

}  // namespace hk

using namespace hk;

static int kdist_common(const double *kappa, int64_t n_points, double dnu, double bin_width, int n_g, double *k_out, int n_c,
                        double *coef_out, void *stream)
{
  if (!kappa || (!k_out && !coef_out) || n_points < 1 || !(dnu > 0.0) || !isfinite(dnu) || !(bin_width > 0.0) || !isfinite(bin_width) ||
      (k_out && (n_g < 1 || n_g > 128)) || (coef_out && (n_c < 1 || n_c > 64)))
    return HK_ERR_INVALID;
  const double ratio = bin_width / dnu;
  const double ppb_d = nearbyint(ratio);
  if (ppb_d < 1.0 || fabs(ratio - ppb_d) > 1e-9 * ppb_d) return HK_ERR_INVALID;
  if (ppb_d > 16384.0) return HK_ERR_UNSUPPORTED;
  const int ppb = (int)ppb_d;
  if (n_points % ppb != 0) return HK_ERR_INVALID;
  const int64_t n_bins = n_points / ppb;
  if (n_bins > 2147483647LL) return HK_ERR_UNSUPPORTED;
  if (coef_out && n_c > ppb) return HK_ERR_INVALID;  // more coefficients than points: the fit is not determined
  KdistArgs a;
  a.kappa = kappa;
  a.k_out = k_out;
  a.ppb = ppb;
  a.n_g = k_out ? n_g : 0;
  a.ln_out = nullptr;
  cudaStream_t st = (cudaStream_t)stream;
  const double *P = nullptr;
  void *ln_buf = nullptr;
  if (coef_out) {
    int rcp = cheb_projection_device(ppb, n_c, &P);
    if (rcp != HK_OK) return rcp;
    rcp = pool_alloc(&ln_buf, (size_t)n_points * sizeof(double), st);
    if (rcp != HK_OK) return rcp;
    a.ln_out = (double *)ln_buf;
  }
  int n = 64;
  while (n < ppb) n <<= 1;
  a.n = n;
  double wts[128];
  int rc = k_out ? hk_gauss_legendre(n_g, a.g, wts) : HK_OK;
  if (rc == HK_OK) {
    if (n <= 256) rc = launch_kdist<2, 128>(a, n_bins, st);        // T = 32 .. 128
    else if (n == 512) rc = launch_kdist<4, 128>(a, n_bins, st);   // T = 128
    else if (n == 1024) rc = launch_kdist<16, 64>(a, n_bins, st);  // T = 64 (7 % faster than 8 x 128; 32 x 32 is slower)
    else rc = launch_kdist<16, 1024>(a, n_bins, st);               // T = 128 .. 1024
  }
  if (rc == HK_OK && coef_out) {
    const size_t cp_bytes = (size_t)(kCpBins + n_c) * (size_t)((ppb < kCpChunk ? ppb : kCpChunk) + 1) * sizeof(double);
    static PerDeviceOnce cp_attr;
    cudaError_t e = cudaSuccess;
    if (cp_attr.run([](int) {
          cudaError_t ea = cudaFuncSetAttribute(cheb_project_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                                (int)((kCpBins + kCpMaxNc) * (kCpChunk + 1) * sizeof(double)));
          return ea == cudaSuccess ? HK_OK : cuda_fail(ea, "cudaFuncSetAttribute(cheb_project_kernel)");
        }) != HK_OK)
      e = cudaErrorUnknown;
    if (e == cudaSuccess) {
      cheb_project_kernel<<<(unsigned)((n_bins + kCpBins - 1) / kCpBins), 128, cp_bytes, st>>>(a.ln_out, P, n_bins, ppb, n_c,
                                                                                                coef_out);
      e = cudaGetLastError();
    }
    if (e != cudaSuccess) rc = cuda_fail(e, "cheb_project_kernel launch");
  }
  pool_free(ln_buf, st);
  return rc;
}

extern "C" int hk_kdist(const double *kappa, int64_t n_points, double dnu, double bin_width, int n_g, double *k_out,
                        void *stream)
{
  if (!k_out) return HK_ERR_INVALID;
  return kdist_common(kappa, n_points, dnu, bin_width, n_g, k_out, 0, nullptr, stream);
}

extern "C" int hk_kdist_cheb(const double *kappa, int64_t n_points, double dnu, double bin_width, int n_c, double *coef_out,
                             int n_g, double *k_out, void *stream)
{
  if (!coef_out) return HK_ERR_INVALID;
  return kdist_common(kappa, n_points, dnu, bin_width, n_g, k_out, n_c, coef_out, stream);
}
