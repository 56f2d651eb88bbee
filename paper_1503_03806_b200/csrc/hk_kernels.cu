// hk_kernels.cu — sm_100a kernels and the C ABI of include/hk.h.
//
// Steps:
//   a1 line_prep_kernel   per line: alpha, gamma (eq. 20), centre shift (eq. 21), S(T) (eq. 18), amplitude, index window
//                         (absolute or relative cutoff), regime balls in index space, packed records
//   a2 (same kernel)      per 256-point block: first line ending / beginning / centred there (lookup tables: a tile's line
//                         range is two reads)
//   a3 voigt_far_kernel   every 32-point group outside a line's 3-point radius (1-/2-/3-point rule) of kappa_j = sum_i amp_i
//                         V_i(nu_j): grid-point-owned register accumulation, persistent CTAs on a tile queue, lines streamed
//                         through a shared-memory ring by 1-D TMA bulk copies completing on mbarriers; FP64 in two shapes
//                         (by list density), or the FP32 variant (template parameters)
//      voigt_near_kernel  every group that touches it (6-point rule, series): one warp per 256-point span works off queues
//                         of uniform items, per-line constants computed once by lane = line; adds to kappa
//   a4                    coalesced kappa store from the far kernel ("without additional write-outs")
//   a5/a6 kdist_kernel    (hk_kdist.cu) per-bin register/shuffle bitonic sort + resampling at Gauss-Legendre nodes
// eq. 20/21 line physics, mixtures and the relative cutoff live in a1 and the host code below;
// Chebyshev resampling and the transmission function in hk_kdist.cu / hk_resample.cu.
#include <cuda_runtime.h>
#include <limits.h>
#include <math.h>
#include <stdint.h>
#include <stdio.h>
#include <string.h>

#include <algorithm>
#include <new>

#include "../../include/hk.h"
#include "hk_internal.h"
#include "hk_voigt.cuh"

namespace hk {

// Index checks compiled in by -DHK_DEBUG_CHECKS (a trap instead of a silent out-of-range access): compute-sanitizer is closed on
// the GPU pool this was developed on, so the GPU test suite is run once per round against such a build (profiles/).
#ifdef HK_DEBUG_CHECKS
#define HK_CHECK(cond) do { if (!(cond)) __trap(); } while (0)
#else
#define HK_CHECK(cond) do { } while (0)
#endif

// ------------------------------------------------------------------------------------------------------
// packed line records (written by a1, streamed by a3): two 16-byte and three 32-byte records per line, structure of
// arrays, so that a chunk of lines is five contiguous 16-byte-aligned spans (one TMA bulk copy each) and a warp that
// classifies 32 lines at once (lane = line) reads the 16-byte meta records without shared-memory bank conflicts.
// ------------------------------------------------------------------------------------------------------
struct __align__(16) MetaA {
  int jlo, jhi;    // inclusive index window of the line (empty if jhi < jlo)
  int j3lo, j3hi;  // "3-ball": the grid points closer to the centre than the 3-point radius (the 6-point rule and the series
                   // live inside it); INT_MAX, INT_MIN if it holds no grid point
};
struct __align__(16) MetaB {
  int j1lo, j1hi;  // likewise the 1-ball (beyond it: 1-point rule with the shifted denominator)
  int j2lo, j2hi;  // and the 2-ball (beyond it: 2-point rule); ball1 contains ball2 contains ball3
};
struct __align__(16) LineBase {
  double nu0, A1, g2, a2;  // centre; amp*gamma/pi; gamma^2; alpha^2
};
struct __align__(16) LineGH2 {
  double e2, f2, A1a2, inv_alpha;  // gamma^2 - alpha^2/2; 2 alpha^2 gamma^2; A1 alpha^2; 1/alpha (0 if alpha == 0)
};
struct __align__(16) LineCore {
  double y, erfcx_y, Acore, inv_y;  // gamma/alpha (>= 1e-200); erfcx(y); amp/(alpha sqrt(pi)); alpha/gamma.  alpha = 0: y = 1e150
};
struct __align__(16) LineNear {
  int jslo, jshi;  // the grid points that take the series (x^2 <= 44.15 - y^2), inside the 3-ball; INT_MAX, INT_MIN if none
  int tiny;        // 1: y < 1e-8, the 6-point rule adds the Gaussian term exp(-x^2) (no wing rule carries it)
  int pad;
};
// FP32 variant: what the far kernel needs of LineBase + LineGH2, in float, and the line centre in grid units split into an
// integer and a fraction so that d = ((j - ci) - cf) dnu carries no cancellation (relative error 2^-24 at any distance)
// Amplitudes span more than the float range (eq. 18's Boltzmann factor alone reaches e^87 in config 4), so A1 = A1m 2^A1e is
// kept split: the far kernel scales the 32 lines it sums in float by the largest exponent among them.
struct __align__(16) LineF32 {
  int ci;                  // the grid point nearest to the centre
  float cf;                // centre - ci in grid units, in [-1/2, 1/2]
  float A1m;               // amp*gamma/pi = A1m * 2^A1e, A1m in [0.5, 1] (0 for a line of zero strength)
  int A1e;                 // INT_MIN for a line of zero strength (does not enter the batch maximum)
  float g2, e2, f2, a2;    // as LineBase / LineGH2
};
static_assert(sizeof(MetaA) == 16 && sizeof(MetaB) == 16 && sizeof(LineBase) == 32 && sizeof(LineGH2) == 32 &&
                  sizeof(LineCore) == 32 && sizeof(LineF32) == 32 && sizeof(LineNear) == 16,
              "record size");
constexpr size_t kBytesPerLine =
    sizeof(MetaA) + sizeof(MetaB) + sizeof(LineBase) + sizeof(LineGH2) + sizeof(LineCore) + sizeof(LineNear);

constexpr double kCLight = 2.99792458e10;   // cm/s
constexpr double kBoltz = 1.380649e-16;     // erg/K
constexpr double kAmu = 1.66053906660e-24;  // g
constexpr double kC2 = 1.4388;              // cm K (BASELINE.json config 4)
constexpr double kT0 = 296.0;               // K

struct PrepArgs {
  const double *nu0, *S, *gamma0, *n_T, *E_low;
  const double *gamma_self, *A21;  // eq. 20 (either may be NULL)
  const double *delta;             // eq. 21 (may be NULL): the centre used downstream is nu0 + delta P
  double shift_pad;                // >= max |delta| P, cm^-1: the a2 tables are built from the UNSHIFTED (ordered) centres with
                                   // the cutoff widened by it, a superset of every shifted line's window
  double self_fraction, abundance;
  double cutoff_widths;  // > 0: line i is truncated at min(cutoff, cutoff_widths * gamma_i)
  int64_t n;
  double T, P_atm, tfac_half;  // (296/T)^0.5 for n_T == NULL
  double vth;                  // sqrt(2 kB T/m)/c : alpha = nu0*vth
  double inv_mg;               // 1/(m*amu)
  double q_ratio;
  double nu_min, dnu, cutoff;
  int N;
  double R2, R3;      // switch radii on r^2 of the 2-, 3-point rule (kR2.. for FP64, kR2f.. for the FP32 variant)
  int f32_ladder;     // the 1-point rule's switch is r1_sq(y, f32_ladder)
  LineF32 *f32;       // FP32 variant only (else NULL)
  MetaA *ma;
  MetaB *mb;
  LineBase *base;
  LineGH2 *gh2;
  LineCore *core;
  LineNear *near;
  int nb;         // number of plan blocks of kPlanBlock grid points, ceil(N / kPlanBlock)
  int *first_hi;  // [nb+1]  first_hi[b] = first line i with jhi_i >= b*kPlanBlock   (n if none)
  int *first_lo;  // [nb+1]  first_lo[b] = first line i with jlo_i >= b*kPlanBlock   (n if none)
  int *first_c;   // [nb+1]  first_c[b]  = first line i centred at or beyond grid point b*kPlanBlock   (n if none)
  int *queue;     // tile-ticket counter of a3, reset here
};

constexpr int kPlanBlock = 256;  // granularity of the line-range lookup and of the cost model of a2

// FP32 variant: half-width, in grid points, of the band around every line centre that the FP64 near kernel serves (line_prep)
__host__ __device__ __forceinline__ double f32_guard_points(double dnu) { return fmax(3.0, ceil(4.0e-5 / dnu)); }

// index window of a line: sub, sub, IEEE divide, ceil/floor — no multiply-add, nothing to contract (A4)
__device__ __forceinline__ void line_window(double nu0, double cutoff, const PrepArgs &a, int &jlo, int &jhi)
{
  double lo = ceil(__ddiv_rn(__dsub_rn(__dsub_rn(nu0, cutoff), a.nu_min), a.dnu));
  double hi = floor(__ddiv_rn(__dsub_rn(__dadd_rn(nu0, cutoff), a.nu_min), a.dnu));
  if (!(lo > 0.0)) lo = 0.0;
  if (!(hi < (double)(a.N - 1))) hi = (double)(a.N - 1);
  if (lo > 2.0e9) lo = 2.0e9;
  if (hi < -2.0e9) hi = -2.0e9;
  jlo = (int)lo;
  jhi = (int)hi;
}
// floor of the line centre in grid units, clamped to the int range (monotone in nu0)
__device__ __forceinline__ int line_centre_index(double nu0, const PrepArgs &a)
{
  const double c = floor((nu0 - a.nu_min) * (1.0 / a.dnu));
  return (int)fmin(fmax(c, -2.0e9), 2.0e9);
}
// floor(j / kPlanBlock) for any sign
__device__ __forceinline__ int plan_block_floor(int j) { return j >> 8; }
static_assert(kPlanBlock == 256, "plan_block_floor shifts by 8");

// The grid points within rho grid steps of the centre c, as an inclusive index range (INT_MAX, INT_MIN if there is none).
// Every regime decision of a3 is taken on such ranges, in integers, by both kernels: a rule is used on a point only when
// the point lies outside the ball the rule is valid beyond.
__device__ __forceinline__ void ball_range(double c, double rho, int &lo, int &hi)
{
  lo = INT_MAX;
  hi = INT_MIN;
  if (!(rho >= 0.0)) return;
  const double l = fmax(ceil(c - rho), -2.0e9), h = fmin(floor(c + rho), 2.0e9);
  if (l > h) return;
  lo = (int)l;
  hi = (int)h;
}
// ... for the ball x^2 + y^2 < R, i.e. |nu - nu0| < sqrt(R alpha^2 - gamma^2) (a hair outward: 1e-9 relative)
__device__ __forceinline__ void ball_of(double R, double a2, double g2, double c, double inv_dnu, int &lo, int &hi)
{
  const double t = R * a2 - g2;
  ball_range(c, t > 0.0 ? sqrt(t) * inv_dnu * (1.0 + 1.0e-9) : -1.0, lo, hi);
}

__global__ void __launch_bounds__(256) line_prep_kernel(PrepArgs a)
{
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= a.n) return;
  if (i < 16) a.queue[i] = 0;  // one ticket counter per far-kernel launch of this call (at most kMaxChunks)
  if (a.n < 16 && i == 0)
    for (int q = (int)a.n; q < 16; ++q) a.queue[q] = 0;
  // eq. 21: nu0 -> nu0 + delta P/P0, P0 = 1 atm; the shifted centre replaces nu0 everywhere downstream
  // (C2).  The list stays in the order of the unshifted centres: nothing below needs the shifted ones ordered.
  const double nu0u = a.nu0[i];
  const double nu0 = a.delta ? __dadd_rn(nu0u, __dmul_rn(a.delta[i], a.P_atm)) : nu0u;
  double alpha = nu0 * a.vth;
  if (!(alpha > 1.0e-290)) alpha = 0.0;  // nu0 <= 0 (or a width whose reciprocal overflows): Lorentzian (A9)
  const double tfac = a.n_T ? pow(kT0 / a.T, a.n_T[i]) : a.tfac_half;
  double gamma;
  if (a.gamma_self) {  // eq. 20: air and self broadening, P0 = 1 atm
    const double P_self = a.self_fraction * a.P_atm;
    gamma = tfac * (a.gamma0[i] * (a.P_atm - P_self) + a.gamma_self[i] * P_self);
  } else {
    gamma = a.gamma0[i] * a.P_atm * tfac;
  }
  if (a.A21) gamma += a.A21[i] * (1.0 / (4.0 * kPi * kCLight));  // natural width
  double S = a.S[i];
  if (a.E_low) {  // eq. 18, PAPER.md:170 (T0 in the last denominator: DESIGN.md G1)
    const double boltz = exp(-kC2 * a.E_low[i] * (1.0 / a.T - 1.0 / kT0));
    const double stim = (nu0 == 0.0) ? kT0 / a.T : (-expm1(-kC2 * nu0 / a.T)) / (-expm1(-kC2 * nu0 / kT0));
    S = S * a.q_ratio * boltz * stim;
  }
  const double amp = S * a.inv_mg * a.abundance;
  const double g2 = gamma * gamma, a2 = alpha * alpha;
  LineBase b;
  b.nu0 = nu0;
  b.A1 = amp * gamma * (1.0 / kPi);
  b.g2 = g2;
  b.a2 = a2;
  LineGH2 g;
  g.e2 = g2 - 0.5 * a2;
  g.f2 = 2.0 * a2 * g2;
  g.A1a2 = b.A1 * a2;
  g.inv_alpha = alpha > 0.0 ? 1.0 / alpha : 0.0;
  LineCore k;
  // gamma = 0 (gamma0 = 0 and no natural width: the pure Doppler limit K(x,0) = exp(-x^2)) is served by the floor on y: every
  // wing rule is then 0 (A1 = 0), the series has sin^2(xy)/y -> 0, and the 6-point rule adds the Gaussian term (y < 1e-8)
  k.y = alpha > 0.0 ? fmax(gamma * g.inv_alpha, 1.0e-200) : 1.0e150;  // series region x^2 < 44 - y^2: none for alpha = 0
  k.inv_y = alpha > 0.0 ? 1.0 / k.y : 0.0;
  k.erfcx_y = core_xc2(k.y) > 0.0 ? erfcx(k.y) : 0.0;
  k.Acore = amp * g.inv_alpha * kInvSqrtPi;
  MetaA ma;
  MetaB mb;
  LineNear nr;
  // relative cutoff, pressure shift: the line's own window is narrower than, or displaced within, the window of the
  // unshifted centre with the absolute cutoff widened by the largest shift; the a2 tables are built from the latter (qlo,
  // qhi: non-decreasing in i, a superset), classify32 masks with the former
  double cut = a.cutoff;
  if (a.cutoff_widths > 0.0) cut = fmin(cut, __dmul_rn(a.cutoff_widths, gamma));
  line_window(nu0, cut, a, ma.jlo, ma.jhi);
  const double tcut = a.cutoff + a.shift_pad;
  int qlo, qhi;
  line_window(nu0u, tcut, a, qlo, qhi);
  {
    // a2, line-parallel half: the list is ordered by nu0, so jlo and jhi are non-decreasing in i and line i is the
    // "first line with jhi >= b*kPlanBlock" exactly for the blocks b with jhi_{i-1} < b*kPlanBlock <= jhi_i (same for jlo).
    // Each entry of first_hi / first_lo has exactly one writer; the last line also fills the blocks beyond its window.
    int plo = INT_MIN, phi = INT_MIN, pc = INT_MIN;
    if (i > 0) {
      line_window(a.nu0[i - 1], tcut, a, plo, phi);
      pc = line_centre_index(a.nu0[i - 1], a);
    }
    const int jc = line_centre_index(nu0u, a);
    const int n = (int)a.n;
    int b0 = i > 0 ? max(plan_block_floor(phi) + 1, 0) : 0, b1 = min(plan_block_floor(qhi), a.nb);
    HK_CHECK(b0 >= 0 && b1 <= a.nb);
    for (int b = b0; b <= b1; ++b) a.first_hi[b] = (int)i;
    if (i == n - 1)
      for (int b = max(plan_block_floor(qhi) + 1, 0); b <= a.nb; ++b) a.first_hi[b] = n;
    b0 = i > 0 ? max(plan_block_floor(plo) + 1, 0) : 0;
    b1 = min(plan_block_floor(qlo), a.nb);
    for (int b = b0; b <= b1; ++b) a.first_lo[b] = (int)i;
    if (i == n - 1)
      for (int b = max(plan_block_floor(qlo) + 1, 0); b <= a.nb; ++b) a.first_lo[b] = n;
    b0 = i > 0 ? max(plan_block_floor(pc) + 1, 0) : 0;
    b1 = min(plan_block_floor(jc), a.nb);
    for (int b = b0; b <= b1; ++b) a.first_c[b] = (int)i;
    if (i == n - 1)
      for (int b = max(plan_block_floor(jc) + 1, 0); b <= a.nb; ++b) a.first_c[b] = n;
  }
  const double inv_dnu = 1.0 / a.dnu;
  const double c = (nu0 - a.nu_min) * inv_dnu;
  // regime balls in index space, nested: series inside ball3 inside ball2 inside ball1
  if (alpha > 0.0) {
    ball_of(r1_sq(k.y, a.f32_ladder != 0), a2, g2, c, inv_dnu, mb.j1lo, mb.j1hi);
    ball_of(a.R2, a2, g2, c, inv_dnu, mb.j2lo, mb.j2hi);
    ball_of(a.R3, a2, g2, c, inv_dnu, ma.j3lo, ma.j3hi);
    const double xs2 = core_xc2(k.y) > 0.0 ? core_xc2(k.y) + kSeriesPad : -1.0;
    ball_range(c, xs2 > 0.0 ? sqrt(xs2) * alpha * inv_dnu : -1.0, nr.jslo, nr.jshi);
    // only the 6-point rule adds the Gaussian term of a tiny-y line: no cheaper rule inside that radius
    const double xg2 = gauss_xg2(k.y);
    nr.tiny = xg2 > 0.0 ? 1 : 0;
    if (xg2 > 0.0) {
      int glo, ghi;
      ball_range(c, sqrt(xg2) * alpha * inv_dnu * (1.0 + 1.0e-9), glo, ghi);
      ma.j3lo = min(ma.j3lo, glo);
      ma.j3hi = max(ma.j3hi, ghi);
    }
    if (a.f32 && a2 < 1.0e-9) {
      // FP32 variant: the float 2-/3-point rules form d^4 and d^6, which leave the float range for a line this narrow
      // (nu0 of a few cm^-1): inside its 1-ball (a fraction of a grid step wide) everything goes to the FP64 near kernel
      mb.j2lo = mb.j1lo; mb.j2hi = mb.j1hi;
      ma.j3lo = mb.j1lo; ma.j3hi = mb.j1hi;
    }
    ma.j3lo = min(ma.j3lo, nr.jslo); ma.j3hi = max(ma.j3hi, nr.jshi);
    mb.j2lo = min(mb.j2lo, ma.j3lo); mb.j2hi = max(mb.j2hi, ma.j3hi);
    mb.j1lo = min(mb.j1lo, mb.j2lo); mb.j1hi = max(mb.j1hi, mb.j2hi);
  } else {
    mb.j1lo = mb.j2lo = ma.j3lo = nr.jslo = INT_MAX;
    mb.j1hi = mb.j2hi = ma.j3hi = nr.jshi = INT_MIN;
    nr.tiny = 0;
  }
  nr.pad = 0;
  if (a.f32) {
    // FP32 variant: the far kernel forms the distance of point j0 + 32k as 32k dnu + d0 in float, which cancels within a few
    // grid steps of the centre (error 1.5e-5 grid steps): the three grid points on either side go to the FP64 near kernel
    // The float 1- and 2-point rules invert a product of denominators ~ d^8 (gh1_acc4f, gh2_acc2p), inside the float range
    // only for 1.8e-5 < |d| < 6.5e4 cm^-1.  Small side: on a grid finer than 1.3e-5 cm^-1 the guard band widens from three grid
    // points to 4e-5 cm^-1 (f32_guard_points, which the near kernel's line search allows for).  Large side: a line whose
    // window reaches beyond 5e4 cm^-1 from its centre (a cutoff that wide, on a list that far from the grid) takes the
    // 3-point rule — one pair of denominators ~ d^6, in range to 2.6e6 cm^-1 — on its whole window; validate() refuses the
    // FP32 variant with a cutoff beyond 2e6 cm^-1.
    int lo3, hi3;
    ball_range(c, f32_guard_points(a.dnu), lo3, hi3);
    ma.j3lo = min(ma.j3lo, lo3); ma.j3hi = max(ma.j3hi, hi3);
    if (ma.jhi >= ma.jlo && fmax((double)ma.jhi - c, c - (double)ma.jlo) * a.dnu > 5.0e4) {
      mb.j2lo = min(mb.j2lo, ma.jlo); mb.j2hi = max(mb.j2hi, ma.jhi);
    }
    mb.j2lo = min(mb.j2lo, ma.j3lo); mb.j2hi = max(mb.j2hi, ma.j3hi);
    mb.j1lo = min(mb.j1lo, mb.j2lo); mb.j1hi = max(mb.j1hi, mb.j2hi);
    LineF32 f;
    const double cc = fmin(fmax(c, -2.0e9), 2.0e9);
    const double cfl = rint(cc);  // nearest: |cf| <= 1/2, so (j - ci) - cf keeps float relative accuracy at the centre too
    f.ci = (int)cfl;
    f.cf = (float)(cc - cfl);
    int ex = 0;
    f.A1m = (float)frexp(b.A1, &ex);
    f.A1e = b.A1 > 0.0 ? ex : INT_MIN;  // a line of zero strength does not raise its batch's scale
    f.g2 = (float)g2; f.e2 = (float)g.e2; f.f2 = (float)g.f2; f.a2 = (float)a2;
    a.f32[i] = f;
  }
  a.ma[i] = ma;
  a.mb[i] = mb;
  a.base[i] = b;
  a.gh2[i] = g;
  a.core[i] = k;
  a.near[i] = nr;
}

// ------------------------------------------------------------------------------------------------------
// mbarrier + 1-D TMA bulk copy (cp.async.bulk -> SASS UBLKCP)
// ------------------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count)
{
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_fence_init()
{
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes)
{
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t *bar)
{
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void *dst, const void *src, uint32_t bytes, uint64_t *bar)
{
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                   smem_u32(dst)),
               "l"(src), "r"(bytes), "r"(smem_u32(bar))
               : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity)
{
  uint32_t ok;
  const uint32_t addr = smem_u32(bar);
#ifdef HK_WATCHDOG
  const long long t0 = clock64();
#endif
  do {
    asm volatile(
        "{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(ok)
        : "r"(addr), "r"(parity)
        : "memory");
#ifdef HK_WATCHDOG
    if (!ok && clock64() - t0 > 4000000000LL) __trap();  // ~2 s: a protocol bug must not hang the GPU
#endif
  } while (!ok);
}

// ------------------------------------------------------------------------------------------------------
// a3 + a4: Voigt accumulation, in two kernels that split the (line, 32-point group) pairs between them by ONE integer
// test: does the group touch the line's 3-ball (MetaA.j3lo..j3hi)?
//
//   voigt_far_kernel   every group that lies wholly outside the 3-ball: 1-, 2- or 3-point Gauss-Hermite rule, chosen per
//                      (line, 256-point span) where the whole span is beyond a ball, per group on the spans that touch
//                      the 3-ball (99.4 % of all evaluations of config 1), and writes kappa;
//   voigt_near_kernel  every group that touches the 3-ball (6-point rule, series), and adds to kappa.
//
// Why two: the far work of a chunk of lines is the same for every warp of a CTA, the near work is not (it falls on the one
// warp whose span holds the line centres; in a dense list, config 3, on the same warp for hundreds of consecutive chunks),
// and warps that share a line ring can drift apart by only STAGES-1 chunks.  Kept apart, the far kernel streams lines through
// a shared ring in lockstep at full rate, and the near kernel works off uniform items (one rule, 32 points) in tight loops.
// Each grid point has one owner per kernel and a fixed summation order: results are bitwise reproducible.
//
// Far kernel.  Persistent CTAs of WARPS warps, all of them consumers.  Work unit = tile of WARPS*32*P consecutive grid
// points, pulled from an atomic queue.  Warp w owns the span [tile_lo + w*32P, +32P), lane l the points span_lo + l + 32k
// (k < P): stores are coalesced, every 32 consecutive points ("group") belong to one k, and a thread carries P independent
// dependency chains.  The lines of the tile's range are streamed through a STAGES-deep shared-memory ring in chunks of CH
// lines: four 1-D TMA bulk copies per chunk (the four record spans) completing on the stage's `full` mbarrier; the last
// warp out of a stage refills it (ticket-ordered).  No CTA-wide barrier exists after start-up, and the ring keeps flowing
// across tile boundaries (each stage carries a header naming its tile).
// A warp handles a chunk 32 lines at a time.  First it CLASSIFIES them, lane = line: integer compares of the span against
// the line's window and balls (from a1) pick the rule valid on the whole span, and ballots turn that into bit masks.  Then
// it walks each mask: a branch-free loop over the lines of one rule, parameters broadcast from shared memory, an unrolled
// P-point body accumulating in registers: ~1 instruction per (line, span) for the regime decision, no divergence.
// ------------------------------------------------------------------------------------------------------
// Shape of a far-kernel instantiation: P points per thread (groups per warp), WARPS warps per CTA sharing one line ring of
// STAGES stages of CH lines, MINB CTAs per SM; F32 = the FP32 variant.
template <int P_, int WARPS_, int MINB_, int CH_, int STAGES_, bool F32_>
struct FarShape {
  static constexpr int P = P_, WARPS = WARPS_, MINB = MINB_, CH = CH_, STAGES = STAGES_;
  static constexpr bool F32 = F32_;
  static constexpr int TILE = WARPS_ * 32 * P_;
};

struct __align__(16) StageHdr {
  int tile_lo;  // first grid point of the tile this chunk belongs to; < 0: no more work
  int cnt;      // lines in the chunk (0 for a tile no line touches)
  int flags;    // 1: first chunk of its tile, 2: last chunk of its tile
  int ws;       // points per warp span in this tile (<= 32 P)
  int tile_hi;  // one past the last grid point of the tile
  int pad[3];
};

template <bool F32, int CH, int STAGES>
struct RingRecs {  // FP64: two 32-byte records per line
  LineBase base[STAGES][CH];
  LineGH2 gh2[STAGES][CH];
  static constexpr uint32_t kBytes = 16u + 16u + 32u + 32u;  // ring bytes per line, with MetaA and MetaB
};
template <int CH, int STAGES>
struct RingRecs<true, CH, STAGES> {  // FP32 variant: one
  LineF32 f32[STAGES][CH];
  static constexpr uint32_t kBytes = 16u + 16u + 32u;
};

template <class Sh>
struct __align__(128) VoigtSmem {
  static constexpr int CH = Sh::CH, STAGES = Sh::STAGES;
  using Recs = RingRecs<Sh::F32, Sh::CH, Sh::STAGES>;
  MetaA ma[STAGES][CH];
  MetaB mb[STAGES][CH];
  Recs r;
  StageHdr hdr[STAGES];
  uint64_t full[STAGES];
  int done[STAGES];  // warps that have finished with the stage's current chunk
  int issued;        // chunks handed to the TMA engine so far (ticket that orders the refills)
  // refill cursor: owned by whoever holds ticket `issued`
  int cur_tile, cur_L0, cur_nl, cur_c, cur_nchunks, cur_stop;
  int descending;  // tiles are handed out from the top of the grid (heavier tiles first)
};

struct VoigtArgs {
  const MetaA *ma;
  const MetaB *mb;
  const LineBase *base;
  const LineGH2 *gh2;
  const LineCore *core;
  const LineNear *near;
  const LineF32 *f32;   // FP32 variant only
  const int *first_hi;  // a2 lookup tables (see PrepArgs)
  const int *first_lo;
  const int *first_c;
  int *queue;           // tile tickets of the far kernel (reset by a1)
  int nb, n_tiles;      // plan blocks of the grid; tiles of THIS far-kernel launch, which start at tile0
  int tile0;
  double nu_min, dnu;
  float dnu_f;
  int N;
  int n_lines;
  int accumulate;  // 1: add to kappa (species of a mixture after the first), 0: overwrite
  int block0;      // near kernel: first 256-point span of this launch (the near kernel may run as several launches)
  double *kappa;
  double r3_slope, r3_offset;  // near kernel: no line centred beyond r3_slope*j + r3_offset grid units of point j has j in its 3-ball
};

// lane = line classification of 32 lines against the 256-point span [slo, shi].  Bit masks of the lines that
//   m1, m2, m3 : take the 1- / 2- / 3-point rule on the whole span, span inside the line's window
//   e1, e2     : 1- / 2-point rule, but a cutoff edge of the line falls inside the span: masked to the window
//   n3         : the rest of the lines that touch the span: 3-point rule on the groups outside the 3-ball, masked to the
//                window (the groups that touch the 3-ball are the near kernel's)
struct SpanMasks {
  unsigned m1, m2, m3, e1, e2, n3;
};
__device__ __forceinline__ SpanMasks classify_regs(const MetaA &A, const MetaB &B, bool live, int slo, int shi)
{
  const bool act = live && (shi >= slo) && (A.jhi >= slo) && (A.jlo <= shi);
  const bool inside = (A.jlo <= slo) && (A.jhi >= shi);
  const bool b1 = (shi < B.j1lo) || (slo > B.j1hi);  // the span lies beyond the 1-ball ...
  const bool b2 = (shi < B.j2lo) || (slo > B.j2hi);
  const bool b3 = (shi < A.j3lo) || (slo > A.j3hi);
  SpanMasks M;
  M.m1 = __ballot_sync(kFull, act && inside && b1);
  M.m2 = __ballot_sync(kFull, act && inside && !b1 && b2);
  M.m3 = __ballot_sync(kFull, act && inside && !b2 && b3);
  M.e1 = __ballot_sync(kFull, act && !inside && b1);
  M.e2 = __ballot_sync(kFull, act && !inside && !b1 && b2);
  M.n3 = __ballot_sync(kFull, act && !b2 && !(inside && b3));
  return M;
}
__device__ __forceinline__ SpanMasks classify32(const MetaA *ma, const MetaB *mb, int l, int cnt, int slo, int shi)
{
  const bool live = l < cnt;
  return classify_regs(ma[live ? l : 0], mb[live ? l : 0], live, slo, shi);
}
// the far kernel's share of a span that touches a line's 3-ball: the 32-point groups [glo, glo+31] wholly outside it
__device__ __forceinline__ bool group_is_far(int glo, int j3lo, int j3hi) { return (glo + 31 < j3lo) || (glo > j3hi); }

// lines that can touch the grid points [lo, hi): jhi >= lo and jlo < hi, looked up at plan-block granularity (a superset
// by at most the lines that end or begin inside the two boundary blocks; classify32 masks them out)
__device__ __forceinline__ int2 tile_lines(const VoigtArgs &a, int lo, int hi)
{
  const int L0 = a.first_hi[lo / kPlanBlock];
  const int L1 = a.first_lo[min((hi + kPlanBlock - 1) / kPlanBlock, a.nb)];
  return make_int2(L0, max(L1, L0));
}

// Hands the next chunk of lines (ring sequence number n) to the TMA engine: stage n % STAGES gets a header and, if the chunk
// holds lines, four bulk copies completing on the stage's `full` mbarrier.  Pulls a new tile from the queue when the current
// one is exhausted; after the last tile one stop header is posted and nothing more.  Called by one thread at a time, in
// order of n (ticket S.issued).
template <class Sh>
__device__ __forceinline__ void issue_chunk(VoigtSmem<Sh> &S, const VoigtArgs &a, int n)
{
  constexpr int TILE = Sh::TILE, CH = Sh::CH, STAGES = Sh::STAGES, P = Sh::P;
  constexpr bool F32 = Sh::F32;
  if (S.cur_stop) return;
  const int stage = n % STAGES;
  if (S.cur_c == S.cur_nchunks) {
    const int ticket = atomicAdd(a.queue, 1);
    if (ticket >= a.n_tiles) {
      S.cur_stop = 1;
      StageHdr h = {};
      h.tile_lo = -1;
      S.hdr[stage] = h;
      mbar_expect_tx(&S.full[stage], 0u);
      return;
    }
    const int tile = a.tile0 + (S.descending ? a.n_tiles - 1 - ticket : ticket);
    const int2 pl = tile_lines(a, tile * TILE, min((tile + 1) * TILE, a.N));
    const int nl = pl.y - pl.x;
    S.cur_tile = tile;
    S.cur_L0 = pl.x;
    S.cur_nl = nl;
    S.cur_c = 0;
    S.cur_nchunks = nl > 0 ? (nl + CH - 1) / CH : 1;
  }
  const int c = S.cur_c;
  const int cnt = min(CH, S.cur_nl - c * CH);
  StageHdr h = {};
  h.tile_lo = S.cur_tile * TILE;
  h.tile_hi = min(h.tile_lo + TILE, a.N);
  h.ws = 32 * P;
  h.cnt = cnt > 0 ? cnt : 0;
  h.flags = (c == 0 ? 1 : 0) | (c == S.cur_nchunks - 1 ? 2 : 0);
  S.hdr[stage] = h;
  S.cur_c = c + 1;
  const uint32_t nb = (uint32_t)h.cnt;
  HK_CHECK(h.cnt >= 0 && h.cnt <= CH && S.cur_L0 >= 0 && S.cur_L0 + c * CH + h.cnt <= a.n_lines && stage >= 0 && stage < STAGES);
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");  // the stage's previous readers (generic proxy) come first
  mbar_expect_tx(&S.full[stage], nb * VoigtSmem<Sh>::Recs::kBytes);  // release: the header store above is visible to the waiters
  if (nb) {
    const int first = S.cur_L0 + c * CH;
    bulk_g2s(&S.ma[stage][0], a.ma + first, nb * 16u, &S.full[stage]);
    bulk_g2s(&S.mb[stage][0], a.mb + first, nb * 16u, &S.full[stage]);
    if constexpr (F32) {
      bulk_g2s(&S.r.f32[stage][0], a.f32 + first, nb * 32u, &S.full[stage]);
    } else {
      bulk_g2s(&S.r.base[stage][0], a.base + first, nb * 32u, &S.full[stage]);
      bulk_g2s(&S.r.gh2[stage][0], a.gh2 + first, nb * 32u, &S.full[stage]);
    }
  }
}

template <class Sh>
__global__ void __launch_bounds__(Sh::WARPS * 32, Sh::MINB) voigt_far_kernel(const __grid_constant__ VoigtArgs a)
{
  constexpr int P = Sh::P, WARPS = Sh::WARPS, STAGES = Sh::STAGES;
  constexpr bool F32 = Sh::F32;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  VoigtSmem<Sh> &S = *reinterpret_cast<VoigtSmem<Sh> *>(smem_raw);

  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  if (threadIdx.x == 0) {
    for (int s = 0; s < STAGES; ++s) {
      mbar_init(&S.full[s], 1);
      S.done[s] = 0;
    }
    S.cur_tile = 0; S.cur_L0 = 0; S.cur_nl = 0; S.cur_c = 0; S.cur_nchunks = 0; S.cur_stop = 0;
    {
      // heavier tiles first: compare the line counts of the first and the last tile
      constexpr int TILE = Sh::TILE;
      const int2 f = tile_lines(a, a.tile0 * TILE, min((a.tile0 + 1) * TILE, a.N)),
                 l = tile_lines(a, (a.tile0 + a.n_tiles - 1) * TILE, min((a.tile0 + a.n_tiles) * TILE, a.N));
      S.descending = (l.y - l.x) >= (f.y - f.x);
    }
    mbar_fence_init();
    for (int n = 0; n < STAGES; ++n) issue_chunk<Sh>(S, a, n);  // fill the ring
    S.issued = STAGES;
  }
  __syncthreads();  // the only CTA-wide barrier

  int slo = 0, shi = -1;  // this warp's span of the current tile, inclusive (empty if shi < slo)
  int stage = 0;
  uint32_t phase = 0;
  double x0 = 0.0;
  double acc[P];  // kappa of this thread's P points, carried in registers over all chunks of a tile
#pragma unroll
  for (int k = 0; k < P; ++k) acc[k] = 0.0;

  for (int n = 0;; ++n) {
    mbar_wait(&S.full[stage], phase);
    const StageHdr h = S.hdr[stage];
    if (h.tile_lo < 0) break;
    if (h.flags & 1) {
      slo = h.tile_lo + warp * h.ws;
      shi = min(slo + h.ws, h.tile_hi) - 1;
      x0 = __dadd_rn(a.nu_min, __dmul_rn((double)(slo + lane), a.dnu));  // nu_j exactly as defined (A6)
    }
    if constexpr (F32) {
      // FP32 variant: float arithmetic, two points per reciprocal.  The 32 lines of a batch are summed in float, with their
      // amplitudes scaled by 2^-eb (eb = largest amplitude exponent of the batch: a line 2^-126 below it flushes to zero,
      // and can nowhere reach 1e-12 of the largest kappa), and the partial sum is added to the FP64 accumulators: the sum over
      // the 1e5 lines that reach a point of config 3 would lose 1e-4 in float alone.
      static_assert(P % 2 == 0, "points are taken in pairs");
      const LineF32 *sf = S.r.f32[stage];
      const int j0 = slo + lane;
#pragma unroll 1
      for (int b0 = 0; b0 < h.cnt; b0 += 32) {
        const SpanMasks M = classify32(S.ma[stage] + b0, S.mb[stage] + b0, lane, h.cnt - b0, slo, shi);
        const unsigned act = M.m1 | M.m2 | M.m3 | M.e1 | M.e2 | M.n3;
        if (act == 0u) continue;
        // (of the lines that contribute to this span only: a strong line of the batch that does not reach it must not flush a
        // weak one that does)
        const int eb = __reduce_max_sync(kFull, ((act >> lane) & 1u) ? sf[b0 + lane].A1e : INT_MIN);
        if (eb == INT_MIN) continue;  // every line of the batch has zero strength
        const int ebm = eb - 127;     // a line more than 2^-127 below the batch maximum flushes to zero
        float af[P];
#pragma unroll
        for (int k = 0; k < P; ++k) af[k] = 0.0f;
        if (M.m1 | M.m2) {
          // whole-span rules on packed pairs of points (k, k+1): FFMA2 / FMUL2 / FADD2, one reciprocal per four (1-point
          // rule) or two (2-point rule) evaluations
          static_assert(P % 4 == 0, "the packed 1-point rule takes four points at a time");
          f32x2 ap[P / 2];
#pragma unroll
          for (int k = 0; k < P / 2; ++k) ap[k] = pk2(0.0f, 0.0f);
#pragma unroll 1
          for (unsigned m = M.m1; m; m &= m - 1) {
            const LineF32 L = sf[b0 + (__ffs(m) - 1)];
            const float w = L.A1m * __int_as_float((max(L.A1e, ebm) - ebm) << 23);
            const float d0 = ((float)(j0 - L.ci) - L.cf) * a.dnu_f;
            const float g2s = fmaf(-1.5f, L.a2, L.g2);
            const f32x2 dd = pk2(d0, d0), gg = pk2(g2s, g2s);
#pragma unroll
            for (int k = 0; k < P / 2; k += 2)
              gh1_acc4f(ap[k], ap[k + 1], add2(dd, pk2((float)(64 * k) * a.dnu_f, (float)(64 * k + 32) * a.dnu_f)),
                        add2(dd, pk2((float)(64 * k + 64) * a.dnu_f, (float)(64 * k + 96) * a.dnu_f)), w, gg);
          }
#pragma unroll 1
          for (unsigned m = M.m2; m; m &= m - 1) {
            const LineF32 L = sf[b0 + (__ffs(m) - 1)];
            const float w = L.A1m * __int_as_float((max(L.A1e, ebm) - ebm) << 23);
            const float d0 = ((float)(j0 - L.ci) - L.cf) * a.dnu_f;
            const float wa2 = w * L.a2;
            const f32x2 dd = pk2(d0, d0), ww = pk2(w, w), ee = pk2(L.e2, L.e2), ff = pk2(L.f2, L.f2), wa = pk2(wa2, wa2);
#pragma unroll
            for (int k = 0; k < P / 2; ++k)
              gh2_acc2p(ap[k], add2(dd, pk2((float)(64 * k) * a.dnu_f, (float)(64 * k + 32) * a.dnu_f)), ww, ee, ff, wa);
          }
#pragma unroll
          for (int k = 0; k < P / 2; ++k) upk2(ap[k], af[2 * k], af[2 * k + 1]);
        }
        // cutoff-edge spans: the same rules, masked to the line's window
#pragma unroll 1
        for (unsigned m = M.e1 | M.e2; m; m &= m - 1) {
          const int i = b0 + (__ffs(m) - 1);
          const bool one = (M.e1 >> (i - b0)) & 1u;
          const int jlo = S.ma[stage][i].jlo, jhi = S.ma[stage][i].jhi;
          const LineF32 L = sf[i];
          const float w = L.A1m * __int_as_float((max(L.A1e, ebm) - ebm) << 23);
          const float d0 = ((float)(j0 - L.ci) - L.cf) * a.dnu_f;
          const float wa2 = w * L.a2;
          const unsigned wlen = (unsigned)(jhi - jlo);
          const int jrel = j0 - jlo;
#pragma unroll
          for (int k = 0; k < P; k += 2) {
            float t0 = 0.0f, t1 = 0.0f;
            const float da = (k == 0 ? d0 : fmaf((float)(32 * k), a.dnu_f, d0)), db = fmaf((float)(32 * k + 32), a.dnu_f, d0);
            if (one) gh1_acc2f(t0, t1, da, db, w, fmaf(-1.5f, L.a2, L.g2));
            else gh2_acc2f(t0, t1, da, db, w, L.e2, L.f2, wa2);
            af[k] += ((unsigned)(jrel + 32 * k) <= wlen) ? t0 : 0.0f;
            af[k + 1] += ((unsigned)(jrel + 32 * k + 32) <= wlen) ? t1 : 0.0f;
          }
        }
        // 3-point rule (float: from r^2 >= 64), whole span / the groups outside the 3-ball, masked to the window
#pragma unroll 1
        for (unsigned m = M.m3 | M.n3; m; m &= m - 1) {
          const int i = b0 + (__ffs(m) - 1);
          const bool whole = (M.m3 >> (i - b0)) & 1u;
          const MetaA A = S.ma[stage][i];
          const LineF32 L = sf[i];
          const float w = L.A1m * __int_as_float((max(L.A1e, ebm) - ebm) << 23);
          const float d0 = ((float)(j0 - L.ci) - L.cf) * a.dnu_f;
          const float e3 = fmaf(-1.5f, L.a2, L.g2), f3 = 3.0f * L.f2;
          const float c3 = w * (1.0f / 3.0f), c0 = 2.0f * c3, c3a = w * L.a2;
          const unsigned wlen = (unsigned)(A.jhi - A.jlo);
          const int jrel = j0 - A.jlo;
#pragma unroll
          for (int k = 0; k < P; ++k) {
            if (whole || group_is_far(slo + 32 * k, A.j3lo, A.j3hi)) {
              const float t = gh3_accf(0.0f, (k == 0 ? d0 : fmaf((float)(32 * k), a.dnu_f, d0)), L.g2, e3, f3, c0, c3, c3a);
              af[k] += ((unsigned)(jrel + 32 * k) <= wlen) ? t : 0.0f;
            }
          }
        }
        const double sc = ldexp(1.0, eb);
#pragma unroll
        for (int k = 0; k < P; ++k) acc[k] = fma((double)af[k], sc, acc[k]);
      }
    } else {
    const LineBase *sbase = S.r.base[stage];
    const LineGH2 *sgh2 = S.r.gh2[stage];
#pragma unroll 1
    for (int b0 = 0; b0 < h.cnt; b0 += 32) {
      const SpanMasks M = classify32(S.ma[stage] + b0, S.mb[stage] + b0, lane, h.cnt - b0, slo, shi);
      // ---- 1-point rule: TWO lines per iteration, four points per reciprocal (gh1_acc4): four independent chains per
      //      thread and half the MUFU.RCP64H of the pair form; measured against one line per iteration with the next line's
      //      record prefetched: config 1 0.807 -> 0.769 ms, config 3 (1e7 lines) 23.4 -> 22.5 ms.  An odd last line is paired
      //      with itself at zero amplitude. ----
      static_assert(P % 4 == 0, "gh1_acc4 takes four points");
#pragma unroll 1
      for (unsigned m = M.m1; m;) {
        const int l0 = __ffs(m) - 1;
        m &= m - 1;
        const bool two = m != 0u;
        const int l1 = two ? __ffs(m) - 1 : l0;
        m &= m - 1;
        const LineBase La = sbase[b0 + l0], Lb = sbase[b0 + l1];
        const double A1a = La.A1, g2a = fma(-1.5, La.a2, La.g2), da = x0 - La.nu0;  // shifted denominator (kR1a)
        const double A1b = two ? Lb.A1 : 0.0, g2b = fma(-1.5, Lb.a2, Lb.g2), db = x0 - Lb.nu0;
#pragma unroll
        for (int k = 0; k < P; k += 4) {
          gh1_acc4(acc[k], acc[k + 1], acc[k + 2], acc[k + 3], (k == 0 ? da : fma((double)(32 * k), a.dnu, da)),
                   fma((double)(32 * k + 32), a.dnu, da), fma((double)(32 * k + 64), a.dnu, da),
                   fma((double)(32 * k + 96), a.dnu, da), A1a, g2a);
          gh1_acc4(acc[k], acc[k + 1], acc[k + 2], acc[k + 3], (k == 0 ? db : fma((double)(32 * k), a.dnu, db)),
                   fma((double)(32 * k + 32), a.dnu, db), fma((double)(32 * k + 64), a.dnu, db),
                   fma((double)(32 * k + 96), a.dnu, db), A1b, g2b);
        }
      }
      // ---- 2-point rule ----
#pragma unroll 1
      for (unsigned m = M.m2; m; m &= m - 1) {
        const int i = b0 + (__ffs(m) - 1);
        const double nu0 = sbase[i].nu0, A1 = sbase[i].A1;
        const double e2 = sgh2[i].e2, f2 = sgh2[i].f2, A1a2 = sgh2[i].A1a2;
        const double d0 = x0 - nu0;
#pragma unroll
        for (int k = 0; k < P; ++k) acc[k] = gh2_acc(acc[k], (k == 0 ? d0 : fma((double)(32 * k), a.dnu, d0)), A1, e2, f2, A1a2);
      }
      // ---- 3-point rule, span wholly between the 3-ball and the 2-ball's edge, inside the window ----
#pragma unroll 1
      for (unsigned m = M.m3; m; m &= m - 1) {
        const LineBase lb = sbase[b0 + (__ffs(m) - 1)];
        const double d0 = x0 - lb.nu0;
        const double e3 = fma(-1.5, lb.a2, lb.g2), f3 = 6.0 * lb.a2 * lb.g2;
        const double c3 = lb.A1 * (1.0 / 3.0), c0 = 2.0 * c3, c3a = lb.A1 * lb.a2;
#pragma unroll
        for (int k = 0; k < P; ++k)
          acc[k] = gh3_acc(acc[k], (k == 0 ? d0 : fma((double)(32 * k), a.dnu, d0)), lb.g2, e3, f3, c0, c3, c3a);
      }
      // ---- the same rules on spans that hold a cutoff edge: masked to the line's window ----
#pragma unroll 1
      for (unsigned m = M.e1; m; m &= m - 1) {
        const int i = b0 + (__ffs(m) - 1);
        const int jlo = S.ma[stage][i].jlo, jhi = S.ma[stage][i].jhi;
        const double nu0 = sbase[i].nu0, A1 = sbase[i].A1, g2 = fma(-1.5, sbase[i].a2, sbase[i].g2);
        const double d0 = x0 - nu0;
        const unsigned wlen = (unsigned)(jhi - jlo);
        const int jrel = slo + lane - jlo;
#pragma unroll
        for (int k = 0; k < P; ++k) {
          const double t = gh1_acc(acc[k], (k == 0 ? d0 : fma((double)(32 * k), a.dnu, d0)), A1, g2);
          acc[k] = ((unsigned)(jrel + 32 * k) <= wlen) ? t : acc[k];
        }
      }
#pragma unroll 1
      for (unsigned m = M.e2; m; m &= m - 1) {
        const int i = b0 + (__ffs(m) - 1);
        const int jlo = S.ma[stage][i].jlo, jhi = S.ma[stage][i].jhi;
        const double nu0 = sbase[i].nu0, A1 = sbase[i].A1;
        const double e2 = sgh2[i].e2, f2 = sgh2[i].f2, A1a2 = sgh2[i].A1a2;
        const double d0 = x0 - nu0;
        const unsigned wlen = (unsigned)(jhi - jlo);
        const int jrel = slo + lane - jlo;
#pragma unroll
        for (int k = 0; k < P; ++k) {
          const double t = gh2_acc(acc[k], (k == 0 ? d0 : fma((double)(32 * k), a.dnu, d0)), A1, e2, f2, A1a2);
          acc[k] = ((unsigned)(jrel + 32 * k) <= wlen) ? t : acc[k];
        }
      }
      // ---- spans that touch the 3-ball (or hold a cutoff edge inside the 2-ball): 3-point rule on the groups wholly
      //      outside the 3-ball (warp-uniform skip), masked to the window; the other groups are the near kernel's ----
#pragma unroll 1
      for (unsigned m = M.n3; m; m &= m - 1) {
        const int i = b0 + (__ffs(m) - 1);
        const MetaA A = S.ma[stage][i];
        const LineBase lb = sbase[i];
        const double d0 = x0 - lb.nu0;
        const double e3 = fma(-1.5, lb.a2, lb.g2), f3 = 6.0 * lb.a2 * lb.g2;
        const double c3 = lb.A1 * (1.0 / 3.0), c0 = 2.0 * c3, c3a = lb.A1 * lb.a2;
        const unsigned wlen = (unsigned)(A.jhi - A.jlo);
        const int jrel = slo + lane - A.jlo;
#pragma unroll
        for (int k = 0; k < P; ++k) {
          if (group_is_far(slo + 32 * k, A.j3lo, A.j3hi)) {
            const double t = gh3_acc(acc[k], (k == 0 ? d0 : fma((double)(32 * k), a.dnu, d0)), lb.g2, e3, f3, c0, c3, c3a);
            acc[k] = ((unsigned)(jrel + 32 * k) <= wlen) ? t : acc[k];
          }
        }
      }
    }
    }  // FP64
    if (h.flags & 2) {  // a4: the tile is complete
#pragma unroll
      for (int k = 0; k < P; ++k) {
        const int j = slo + lane + 32 * k;
        HK_CHECK(j > shi || (j >= 0 && j < a.N));
        if (j <= shi) a.kappa[j] = a.accumulate ? a.kappa[j] + acc[k] : acc[k];
        acc[k] = 0.0;
      }
    }
    // ---- release the stage; the last warp out refills it (ring sequence number n + STAGES), in ticket order ----
    __syncwarp();
    if (lane == 0) {
      __threadfence_block();
      const int old = atomicAdd(&S.done[stage], 1);
      if (old == WARPS - 1) {
        volatile int *issued = &S.issued;
        S.done[stage] = 0;
#ifdef HK_WATCHDOG
        const long long t0 = clock64();
#endif
        while (*issued != n + STAGES) {
#ifdef HK_WATCHDOG
          if (clock64() - t0 > 4000000000LL) __trap();
#endif
        }
        __threadfence_block();
        issue_chunk<Sh>(S, a, n + STAGES);
        __threadfence_block();
        *issued = n + STAGES + 1;
      }
    }
    if (++stage == STAGES) {
      stage = 0;
      phase ^= 1u;
    }
  }
}

// Near kernel.  CTA = one warp = one 256-point span (a plan block); lane l on the points plo + l + 32k of group k.
// The warp walks the lines centred within the span's bound on the 3-ball radius (a2 table first_c) 32 at a time, lane = line:
// a lane whose line has groups of this span inside its 3-ball (and inside its window) computes everything that depends on
// the line alone — the constants of the 6-point rule, the 16 series weights W_n and the folded series constants — ONCE, into
// a shared-memory slot, and writes the line's work as uniform ITEMS into queues:
//   6-point items  (line), one queue per group k of the span: the group's points that are in the window and outside the
//                  series interval; a queue is summed in registers and added to the strip once;
//   series items   (line, first point, count <= 32): chunks of the series interval [jslo, jshi] taken from ITS lower end, not
//                  from the group grid, so that only the last chunk of a line has idle lanes.
// Then the warp works the queues off, two items per iteration (two independent dependency chains per thread), each item one
// rule on 32 points with its constants broadcast from shared memory: no divergence, no per-point rule choice, no constants
// recomputed per group.  Sums are kept in a shared-memory strip that starts as the kappa the far kernel wrote (fetched by
// cp.async while the lines are being listed) and is stored back at the end; order of summation is fixed.
constexpr int kNearP = kPlanBlock / 32;
constexpr int kNearCap = 32;  // lines per round: one per lane
#ifndef HK_NEAR_MINB
#define HK_NEAR_MINB 16
#endif

struct __align__(16) NearSmem {
  double sk[kPlanBlock];
  double W[kNearCap][kTerms];
  double g6[kNearCap][12];  // e, f, cE, c0 of the three +-t pairs
  double nu0[kNearCap];
  SeriesLine ser[kNearCap];  // 5 doubles
  double Acore[kNearCap];
  int4 win[kNearCap];        // jlo, jhi - jlo + 1, jslo, jshi - jslo + 1 (0: no series points): two unsigned range tests
  unsigned int qs[kNearCap * (kNearP + 1) + 2];  // + 2: the series loop prefetches one pair of entries past the last item
  unsigned char q6[kNearP][kNearCap];  // slot | tiny << 5; the items whose group needs no per-point test come first
  int n6[kNearP];
  int n6i[kNearP];                     // how many of them need no test
};

__device__ __forceinline__ void cp_async8(void *smem_dst, const void *gmem_src)
{
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(smem_u32(smem_dst)), "l"(gmem_src) : "memory");
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }

// one 6-point item: line slot u & 31 (bit 5: the line adds the Gaussian term) on the group whose point of this lane is j, at
// nu = xk; 0 outside the window and inside the series interval
template <bool TEST = true>
__device__ __forceinline__ double near_gh6_item(const NearSmem &S, unsigned u, int j, double xk)
{
  const int e = u & 31;
  const double d = xk - S.nu0[e];
  const double *c = S.g6[e];
  const double2 c0 = *reinterpret_cast<const double2 *>(c), c1 = *reinterpret_cast<const double2 *>(c + 2),
                c2 = *reinterpret_cast<const double2 *>(c + 4), c3 = *reinterpret_cast<const double2 *>(c + 6),
                c4 = *reinterpret_cast<const double2 *>(c + 8), c5 = *reinterpret_cast<const double2 *>(c + 10);
  Gh6 G;
  G.p0.e = c0.x; G.p0.f = c0.y; G.p0.cE = c1.x; G.p0.c0 = c1.y;
  G.p1.e = c2.x; G.p1.f = c2.y; G.p1.cE = c3.x; G.p1.c0 = c3.y;
  G.p2.e = c4.x; G.p2.f = c4.y; G.p2.cE = c5.x; G.p2.c0 = c5.y;
  const double q = d * d;
  double v = gh6_val(q, G);
  if (u & 32u) {  // warp-uniform: y < 1e-8, the Gaussian term is still visible beyond the series region
    const double ia = S.ser[e].inv_alpha;
    v = fma(S.Acore[e], exp_fast(fmax(-(q * ia) * ia, -700.0)), v);
  }
  if constexpr (TEST) {
    const int4 w = S.win[e];
    const bool ok = ((unsigned)(j - w.x) < (unsigned)w.y) & !((unsigned)(j - w.z) < (unsigned)w.w);
    return ok ? v : 0.0;
  } else {
    return v;  // the whole group lies in the window and outside the series interval (decided at listing time)
  }
}

__global__ void __launch_bounds__(32, HK_NEAR_MINB) voigt_near_kernel(const __grid_constant__ VoigtArgs a)
{
  __shared__ NearSmem S;
  const int lane = threadIdx.x;
  // spans from the top of the launch's range down: lines widen with wavenumber, so the heavier spans start first and the
  // light ones fill the tail
  const int b = a.block0 + ((int)gridDim.x - 1 - (int)blockIdx.x);
  const int plo = b * kPlanBlock, phi = min(plo + kPlanBlock, a.N) - 1;
  // lines that can have a point of this span in their 3-ball: centre within R of it, and window touching it
  const double R = fmax(fma(a.r3_slope, (double)phi, a.r3_offset), 4.0);
  const double clo = (double)plo - R, chi = (double)phi + R;
  int L0 = a.first_hi[b], L1 = a.first_lo[min(b + 1, a.nb)];
  if (clo > 0.0) L0 = max(L0, a.first_c[min((int)(clo * (1.0 / kPlanBlock)), a.nb)]);
  if (chi < (double)a.nb * kPlanBlock - 1.0) L1 = min(L1, a.first_c[min((int)(chi * (1.0 / kPlanBlock)) + 1, a.nb)]);
  if (L1 <= L0) return;

  // the strip starts as the far kernel's kappa: in flight while the lines are listed
#pragma unroll
  for (int k = 0; k < kNearP; ++k) {
    const int j = plo + 32 * k + lane;
    if (j <= phi) cp_async8(&S.sk[32 * k + lane], a.kappa + j);
    else S.sk[32 * k + lane] = 0.0;
  }
  const double x0 = __dadd_rn(a.nu_min, __dmul_rn((double)(plo + lane), a.dnu));
  bool any = false;

  for (int base0 = L0; base0 < L1; base0 += 32) {
    // ---- lane = line: which groups of the span are this kernel's, per-line constants, items ----
    const int i = base0 + lane;
    const bool live = i < L1;
    const MetaA A = a.ma[live ? i : L0];
    int kA = 1, kB = 0;  // groups that touch the 3-ball and the window (each on its own: the far kernel's test is on the ball alone)
    if (live && A.jhi >= plo && A.jlo <= phi && A.j3hi >= plo && A.j3lo <= phi) {
      kA = (max(max(A.j3lo, A.jlo), plo) - plo) >> 5;
      kB = (min(min(A.j3hi, A.jhi), phi) - plo) >> 5;
    }
    const bool listed = kA <= kB;
    const unsigned lm = __ballot_sync(kFull, listed);
    if (lm == 0u) continue;
    const unsigned lt = (1u << lane) - 1u;
    const int e = __popc(lm & lt);  // slot
    HK_CHECK(!listed || (e < kNearCap && kA >= 0 && kB < kNearP && i < a.n_lines));
    int ns = 0, kS0 = 8, kS1 = -1, sa = 0, sb = -1, sa0 = 0, sb0 = -1;
    unsigned tiny = 0u;
    if (listed) {
      const LineBase lb = a.base[i];
      const LineCore lc = a.core[i];
      const LineNear ln = a.near[i];
      const double inv_alpha = a.gh2[i].inv_alpha;
      sa0 = max(ln.jslo, plo + 32 * kA);  // series points in these groups
      sb0 = min(ln.jshi, plo + 32 * kB + 31);
      if (sa0 <= sb0) {
        kS0 = (sa0 - plo + 31) >> 5;  // groups wholly inside the series interval: no 6-point item
        kS1 = ((sb0 - plo + 1) >> 5) - 1;
        sa = max(sa0, A.jlo);
        sb = min(sb0, A.jhi);
      }
      ns = sb >= sa ? ((sb - sa) >> 5) + 1 : 0;
      tiny = ln.tiny ? 32u : 0u;
      S.nu0[e] = lb.nu0;
      S.Acore[e] = lc.Acore;
      S.win[e] = make_int4(A.jlo, A.jhi - A.jlo + 1, ln.jslo <= ln.jshi ? ln.jslo : 0, ln.jslo <= ln.jshi ? ln.jshi - ln.jslo + 1 : 0);
      if ((kB - kA + 1) > max(kS1 - kS0 + 1, 0)) {
        const Gh6 G = gh6_consts(lb.A1, lb.g2, lb.a2);
        double *c = S.g6[e];
        *reinterpret_cast<double2 *>(c) = make_double2(G.p0.e, G.p0.f);
        *reinterpret_cast<double2 *>(c + 2) = make_double2(G.p0.cE, G.p0.c0);
        *reinterpret_cast<double2 *>(c + 4) = make_double2(G.p1.e, G.p1.f);
        *reinterpret_cast<double2 *>(c + 6) = make_double2(G.p1.cE, G.p1.c0);
        *reinterpret_cast<double2 *>(c + 8) = make_double2(G.p2.e, G.p2.f);
        *reinterpret_cast<double2 *>(c + 10) = make_double2(G.p2.cE, G.p2.c0);
      }
      if (ns > 0) S.ser[e] = series_line_setup(lc.y, lc.inv_y, lc.erfcx_y, lc.Acore, inv_alpha, S.W[e]);
      else S.ser[e].inv_alpha = inv_alpha;  // the Gaussian term of a tiny-y line reads it
    }
    // 6-point queues, one per group: ballot = the lines with an item there, in line order
#pragma unroll
    for (int k = 0; k < kNearP; ++k) {
      const bool has = listed && k >= kA && k <= kB && (k < kS0 || k > kS1);
#ifndef HK_NEAR_NOSPLIT
      // a group wholly inside the line's window that holds no series point needs no per-point test: those items are queued
      // first and worked off by a loop without the test (most items: a window is +-cutoff wide, the 3-ball a few groups)
      const int g0 = plo + 32 * k;
      const bool inner = has && A.jlo <= g0 && A.jhi >= g0 + 31 && (sa0 > sb0 || sb0 < g0 || sa0 > g0 + 31);
      const unsigned bi = __ballot_sync(kFull, inner), be = __ballot_sync(kFull, has && !inner);
      const int ni = __popc(bi);
      HK_CHECK(ni + __popc(be) <= kNearCap);
      if (has) S.q6[k][inner ? __popc(bi & lt) : ni + __popc(be & lt)] = (unsigned char)((unsigned)e | tiny);
      if (lane == 0) {
        S.n6[k] = ni + __popc(be);
        S.n6i[k] = ni;
      }
#else
      const unsigned bk = __ballot_sync(kFull, has);
      HK_CHECK(__popc(bk) <= kNearCap);
      if (has) S.q6[k][__popc(bk & lt)] = (unsigned char)((unsigned)e | tiny);
      if (lane == 0) { S.n6[k] = __popc(bk); S.n6i[k] = 0; }
#endif
    }
    // series queue: exclusive scan of the chunk counts over the lanes
    int incl = ns;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const int t = __shfl_up_sync(kFull, incl, o);
      if (lane >= o) incl += t;
    }
    const int nstot = __shfl_sync(kFull, incl, 31);
    {
      int os = incl - ns;
      for (int j = sa; j <= sb; j += 32) {
        HK_CHECK(os < kNearCap * (kNearP + 1) && j >= plo && j - plo < kPlanBlock && min(sb, j + 31) <= phi);
        S.qs[os++] = (unsigned)e | ((unsigned)(j - plo) << 8) | ((unsigned)(min(sb - j, 31)) << 16);
      }
    }
    if (!any) cp_async_wait_all();
    any = true;
    __syncwarp();

    // ---- 6-point items, group by group, two per iteration, summed in registers ----
#pragma unroll 1
    for (int k = 0; k < kNearP; ++k) {
      const int n = S.n6[k];
      if (n == 0) continue;
      const double xk = fma((double)(32 * k), a.dnu, x0);
      const int j = plo + 32 * k + lane;
      const unsigned char *q = S.q6[k];
      double s0 = 0.0, s1 = 0.0;
      int it = 0;
      const int ni = S.n6i[k] & ~1;  // pairs of untested items; an odd one out goes through the tested loop (same value)
      unsigned nxt = *reinterpret_cast<const unsigned short *>(q);
#pragma unroll 1
      for (; it < ni; it += 2) {
        const unsigned u = nxt;
        nxt = *reinterpret_cast<const unsigned short *>(q + ((it + 2) & 31));
        s0 += near_gh6_item<false>(S, u & 255u, j, xk);
        s1 += near_gh6_item<false>(S, u >> 8, j, xk);
      }
#pragma unroll 1
      for (; it + 1 < n; it += 2) {
        const unsigned u = nxt;
        nxt = *reinterpret_cast<const unsigned short *>(q + ((it + 2) & 31));
        s0 += near_gh6_item(S, u & 255u, j, xk);
        s1 += near_gh6_item(S, u >> 8, j, xk);
      }
      if (it < n) s0 += near_gh6_item(S, nxt & 255u, j, xk);
      S.sk[32 * k + lane] += s0 + s1;
    }
    __syncwarp();
    // ---- series items, two per iteration: point-aligned, so the strip entries of two items may belong to different
    //      lanes: the additions are ordered by __syncwarp ----
    {
      int it = 0;
      uint2 nxt = *reinterpret_cast<const uint2 *>(S.qs);
#pragma unroll 1
      for (; it + 1 < nstot; it += 2) {
        const unsigned u0 = nxt.x, u1 = nxt.y;
        nxt = *reinterpret_cast<const uint2 *>(S.qs + it + 2);
        const int e0 = u0 & 31, e1 = u1 & 31, off0 = (u0 >> 8) & 255, off1 = (u1 >> 8) & 255;
        const double d0 = fma((double)off0, a.dnu, x0) - S.nu0[e0], d1 = fma((double)off1, a.dnu, x0) - S.nu0[e1];
        const SeriesLine Ls0 = S.ser[e0], Ls1 = S.ser[e1];
        const double v0 = series_val(d0, Ls0, S.W[e0]);
        const double v1 = series_val(d1, Ls1, S.W[e1]);
        HK_CHECK(off0 + (int)(u0 >> 16) < kPlanBlock && off1 + (int)(u1 >> 16) < kPlanBlock && (u0 >> 16) < 32u && (u1 >> 16) < 32u);
        if (lane <= (int)(u0 >> 16)) S.sk[off0 + lane] += v0;
        __syncwarp();
        if (lane <= (int)(u1 >> 16)) S.sk[off1 + lane] += v1;
        __syncwarp();
      }
      if (it < nstot) {
        const unsigned u0 = nxt.x;
        const int e0 = u0 & 31, off0 = (u0 >> 8) & 255;
        const double d0 = fma((double)off0, a.dnu, x0) - S.nu0[e0];
        const SeriesLine Ls0 = S.ser[e0];
        const double v0 = series_val(d0, Ls0, S.W[e0]);
        if (lane <= (int)(u0 >> 16)) S.sk[off0 + lane] += v0;
      }
    }
    __syncwarp();  // the slots and queues are free again
  }
  if (!any) return;
#pragma unroll
  for (int k = 0; k < kNearP; ++k) {
    const int j = plo + 32 * k + lane;
    if (j <= phi) a.kappa[j] = S.sk[32 * k + lane];
  }
}

// test hook: out = K(x,y) through the same device functions and switches (alpha = 1, gamma = y, amp = sqrt(pi))
template <bool F32>
__global__ void __launch_bounds__(128) voigt_K_kernel(const double *x, const double *y, int64_t n, double *out)
{
  constexpr double R2 = F32 ? kR2f : kR2, R3 = F32 ? kR3f : kR3;
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const bool live = i < n;
  const double xi = live ? fabs(x[i]) : 1.0e3, yi = live ? fmax(y[i], 1.0e-200) : 1.0;
  const double A1 = yi * kInvSqrtPi;  // amp*gamma/pi with amp = sqrt(pi)  =>  amp*V = K
  const double g2 = yi * yi, a2 = 1.0, q = xi * xi;
  const double r2 = q + g2;
  double v;
  const bool tiny_gauss = q < gauss_xg2(yi);  // only the 6-point branch adds the Gaussian term (as line_prep arranges)
  const double xc2 = core_xc2(yi);
  if (xc2 > 0.0 && q <= xc2 + kSeriesPad) {  // the series interval of a1
    double W[kTerms];
    const SeriesLine L = series_line_setup(yi, 1.0 / yi, erfcx(yi), 1.0, 1.0, W);
    v = series_val(xi, L, W);
  } else if (r2 >= r1_sq(yi, F32) && !tiny_gauss) {
    if constexpr (F32) {  // the far kernel's float arithmetic; the partner point of the pair is a dummy
      float v0 = 0.0f, v1 = 0.0f;
      gh1_acc2f(v0, v1, (float)xi, 1.0f, (float)A1, fmaf(-1.5f, (float)a2, (float)g2));
      v = (double)v0;
    } else {
      v = gh1_acc(0.0, xi, A1, fma(-1.5, a2, g2));
    }
  } else if (r2 >= R2 && !tiny_gauss) {
    if constexpr (F32) {
      float v0 = 0.0f, v1 = 0.0f;
      gh2_acc2f(v0, v1, (float)xi, 1.0f, (float)A1, (float)(g2 - 0.5 * a2), (float)(2.0 * a2 * g2), (float)(A1 * a2));
      v = (double)v0;
    } else {
      v = gh2_acc(0.0, xi, A1, g2 - 0.5 * a2, 2.0 * a2 * g2, A1 * a2);
    }
  } else if (r2 >= R3 && !tiny_gauss) {
    if constexpr (F32) {
      const float c3 = (float)A1 * (1.0f / 3.0f), g2f = (float)g2, a2f = (float)a2;
      v = (double)gh3_accf(0.0f, (float)xi, g2f, fmaf(-1.5f, a2f, g2f), 3.0f * (float)(2.0 * a2 * g2), 2.0f * c3, c3,
                           (float)A1 * a2f);
    } else {
      const double c3 = A1 * (1.0 / 3.0);
      v = gh3_acc(0.0, xi, g2, g2 - 1.5 * a2, 6.0 * a2 * g2, 2.0 * c3, c3, A1 * a2);
    }
  } else {
    v = gh6_val(q, gh6_consts(A1, g2, a2));
    if (tiny_gauss) v += exp_fast(fmax(-q, -700.0));
  }
  if (live) out[i] = v;
}

// largest |delta| of a line list (eq. 21): one atomicMax on the bit pattern of a non-negative double per CTA
__global__ void __launch_bounds__(256) absmax_kernel(const double *v, int64_t n, unsigned long long *out)
{
  double m = 0.0;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) m = fmax(m, fabs(v[i]));
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) m = fmax(m, __shfl_xor_sync(kFull, m, o));
  if ((threadIdx.x & 31) == 0 && m > 0.0) atomicMax(out, (unsigned long long)__double_as_longlong(m));
}

__global__ void __launch_bounds__(256) check_sorted_kernel(const double *nu0, int64_t n, int *flag)
{
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i + 1 < n && !(nu0[i] <= nu0[i + 1])) *flag = 1;
}

__global__ void __launch_bounds__(256) dfma_peak_kernel(double *out, int iters, double a, double b)
{
  double v[8];
#pragma unroll
  for (int i = 0; i < 8; ++i) v[i] = threadIdx.x * 1e-3 + i;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int i = 0; i < 8; ++i) v[i] = fma(v[i], a, b);
  }
  double s = 0.0;
#pragma unroll
  for (int i = 0; i < 8; ++i) s += v[i];
  if (s == 123.456) out[0] = s;
}

__global__ void __launch_bounds__(256) ffma_peak_kernel(float *out, int iters, float a, float b)
{
  float v[16];
#pragma unroll
  for (int i = 0; i < 16; ++i) v[i] = threadIdx.x * 1e-3f + i;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int i = 0; i < 16; ++i) v[i] = fmaf(v[i], a, b);
  }
  float s = 0.0f;
#pragma unroll
  for (int i = 0; i < 16; ++i) s += v[i];
  if (s == 123.456f) out[0] = s;
}

// ------------------------------------------------------------------------------------------------------
// host side
// ------------------------------------------------------------------------------------------------------
static thread_local char g_cuda_err[256] = "";
static thread_local float g_stage_ms[3] = {0.f, 0.f, 0.f};
static thread_local cudaEvent_t g_ev[4] = {nullptr, nullptr, nullptr, nullptr};  // stage boundaries of the last timed call
static thread_local bool g_ev_pending = false;
static thread_local int g_timing = 0;  // per host thread, like the events it fills

int cuda_fail(cudaError_t e, const char *what)
{
  snprintf(g_cuda_err, sizeof(g_cuda_err), "%s: %s", what, cudaGetErrorString(e));
  return e == cudaErrorMemoryAllocation ? HK_ERR_NOMEM : HK_ERR_CUDA;
}
#define HK_CUDA(call)                                  \
  do {                                                 \
    cudaError_t e_ = (call);                           \
    if (e_ != cudaSuccess) return cuda_fail(e_, #call); \
  } while (0)

static bool pos_finite(double v) { return v > 0.0 && isfinite(v); }

// the library's own stream-ordered memory pool, one per device (hk_internal.h)
static int lib_pool(cudaMemPool_t *out)
{
  static cudaMemPool_t pools[64] = {};
  static PerDeviceOnce once;
  int dev = 0;
  HK_CUDA(cudaGetDevice(&dev));
  if (dev < 0 || dev >= 64) return HK_ERR_UNSUPPORTED;
  const int rc = once.run([](int d) {
    cudaMemPoolProps props = {};
    props.allocType = cudaMemAllocationTypePinned;
    props.handleTypes = cudaMemHandleTypeNone;
    props.location.type = cudaMemLocationTypeDevice;
    props.location.id = d;
    cudaMemPool_t mp = nullptr;
    HK_CUDA(cudaMemPoolCreate(&mp, &props));
    uint64_t keep = UINT64_MAX;  // scratch freed by one call is reused by the next; hk_trim() hands it back to the driver
    HK_CUDA(cudaMemPoolSetAttribute(mp, cudaMemPoolAttrReleaseThreshold, &keep));
    pools[d] = mp;
    return (int)HK_OK;
  });
  if (rc != HK_OK) return rc;
  *out = pools[dev];
  return HK_OK;
}
int pool_alloc(void **p, size_t bytes, cudaStream_t st)
{
  *p = nullptr;
  cudaMemPool_t mp = nullptr;
  int rc = lib_pool(&mp);
  if (rc != HK_OK) return rc;
  HK_CUDA(cudaMallocFromPoolAsync(p, bytes ? bytes : 16, mp, st));
  return HK_OK;
}
void pool_free(void *p, cudaStream_t st)
{
  if (p) cudaFreeAsync(p, st);
}

// Far-kernel shapes (measured, profiles/r02_README.md).  4 warps sharing a deep ring (4 x 128 lines) on 1024-point tiles, 4
// CTAs/SM, serve lists up to config 2's density best.  In a very dense list (config 3: 1e5 consecutive lines centred in the same
// 256-point span) the 3-point work of those lines falls on one warp of the four for hundreds of chunks while the others wait at
// the ring: there one warp per CTA with a ring of its own (2 x 64 lines) on 256-point tiles, 16 CTAs/SM, is 9 % faster
// (config 3 at 1e8 lines: far kernel 284 -> 234 ms); on config 1 it is 3 % slower, on config 2 / 4 1-2 % slower over the
// pressure sweep.  The FP32 variant (80 registers) runs one warp per CTA, 24 CTAs/SM, everywhere (16 % faster on config 3).
using ShSparse = FarShape<8, 4, 4, 128, 4, false>;
#ifndef HK_DENSE_WARPS
#define HK_DENSE_WARPS 1
#define HK_DENSE_MINB 16
#define HK_DENSE_CH 64
#define HK_DENSE_STAGES 2
#endif
using ShDense = FarShape<8, HK_DENSE_WARPS, HK_DENSE_MINB, HK_DENSE_CH, HK_DENSE_STAGES, false>;
using ShF32 = FarShape<8, 1, 24, 64, 2, true>;
constexpr double kDenseLinesPerSpan = 10000.0;  // lines whose window reaches a 256-point span, on average, from which ShDense serves

struct Scratch {
  MetaA *ma = nullptr;  // one allocation: ma | mb | base | gh2 | core | near, n_lines records each
  MetaB *mb = nullptr;
  LineBase *base = nullptr;
  LineGH2 *gh2 = nullptr;
  LineCore *core = nullptr;
  LineNear *near = nullptr;
  LineF32 *f32 = nullptr;    // FP32 variant only (same allocation, after near)
  int *first_hi = nullptr;   // one allocation: first_hi[nb+1] | first_lo[nb+1] | first_c[nb+1] | queue
  int *first_lo = nullptr;
  int *first_c = nullptr;
  int *queue = nullptr;
  int64_t cap_lines = 0;
  int cap_blocks = 0;
};

static int scratch_reserve(Scratch &s, int64_t n_lines, int nb, bool f32, cudaStream_t st)
{
  if (n_lines > s.cap_lines || (f32 && !s.f32)) {
    pool_free(s.ma, st);
    s.ma = nullptr; s.f32 = nullptr; s.cap_lines = 0;
    const size_t n = (size_t)n_lines;
    void *p = nullptr;
    int rc = pool_alloc(&p, n * (kBytesPerLine + (f32 ? sizeof(LineF32) : 0)), st);
    if (rc != HK_OK) return rc;
    if (f32) s.f32 = (LineF32 *)((char *)p + n * kBytesPerLine);
    s.ma = (MetaA *)p;
    s.mb = (MetaB *)((char *)p + n * 16);
    s.base = (LineBase *)((char *)p + n * 32);
    s.gh2 = (LineGH2 *)((char *)p + n * 64);
    s.core = (LineCore *)((char *)p + n * 96);
    s.near = (LineNear *)((char *)p + n * 128);
    s.cap_lines = n_lines;
  }
  if (nb > s.cap_blocks) {
    pool_free(s.first_hi, st);
    s.first_hi = nullptr; s.cap_blocks = 0;
    void *p = nullptr;
    int rc = pool_alloc(&p, ((size_t)3 * (nb + 1) + 16) * sizeof(int), st);
    if (rc != HK_OK) return rc;
    s.first_hi = (int *)p;
    s.first_lo = s.first_hi + (nb + 1);
    s.first_c = s.first_lo + (nb + 1);
    s.queue = s.first_c + (nb + 1);
    s.cap_blocks = nb;
  }
  return HK_OK;
}

static void scratch_release(Scratch &s, cudaStream_t st)
{
  pool_free(s.ma, st);
  pool_free(s.first_hi, st);
  s = Scratch();
}

// persistent grid of a3: CTAs resident per SM x SMs of the current device (queried once per device)
template <class Sh>
static int far_grid_of(int dev, int *out)
{
  int sms = 0, per_sm = 0;
  HK_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  HK_CUDA(cudaFuncSetAttribute(voigt_far_kernel<Sh>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(VoigtSmem<Sh>)));
  HK_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, voigt_far_kernel<Sh>, Sh::WARPS * 32, sizeof(VoigtSmem<Sh>)));
  *out = sms * (per_sm < 1 ? 1 : per_sm);
  return HK_OK;
}
// persistent grids of a3: CTAs resident per SM x SMs of the current device, per shape (queried once per device)
enum { kShapeSparse = 0, kShapeDense = 1, kShapeF32 = 2 };
static int voigt_grid(int shape, int *grid_out)
{
  static int grids[64][3] = {};
  static PerDeviceOnce once;
  int dev = 0;
  HK_CUDA(cudaGetDevice(&dev));
  if (dev < 0 || dev >= 64) return HK_ERR_UNSUPPORTED;
  const int rc = once.run([](int d) {
    int rc2 = far_grid_of<ShSparse>(d, &grids[d][kShapeSparse]);
    if (rc2 == HK_OK) rc2 = far_grid_of<ShDense>(d, &grids[d][kShapeDense]);
    if (rc2 == HK_OK) rc2 = far_grid_of<ShF32>(d, &grids[d][kShapeF32]);
    return rc2;
  });
  if (rc != HK_OK) return rc;
  *grid_out = grids[dev][shape];
  return HK_OK;
}

static int validate(const hk_lines *lines, int64_t n_lines, double T, double P_atm, double nu_min, double nu_max, double dnu,
                    double cutoff, const double *kappa_out, const hk_params *prm, int64_t *N_out)
{
  if (!lines || !prm || !kappa_out || n_lines < 0) return HK_ERR_INVALID;
  if (n_lines > 0 && (!lines->nu0 || !lines->S || !lines->gamma0)) return HK_ERR_INVALID;
  if (n_lines > 2000000000LL) return HK_ERR_UNSUPPORTED;
  if (!pos_finite(T) || !pos_finite(P_atm) || !pos_finite(dnu) || !pos_finite(cutoff) || !pos_finite(prm->mass_amu))
    return HK_ERR_INVALID;
  if (!isfinite(nu_min) || !isfinite(nu_max)) return HK_ERR_INVALID;
  if (prm->precision != HK_FP64 && prm->precision != HK_FP32) return HK_ERR_INVALID;
  if (prm->precision == HK_FP32 && cutoff > 2.0e6) return HK_ERR_UNSUPPORTED;  // float range of the wing rules (line_prep)
  if (lines->E_low && !pos_finite(prm->q_ratio)) return HK_ERR_INVALID;
  if (!(prm->abundance >= 0.0) || !isfinite(prm->abundance)) return HK_ERR_INVALID;
  if (!(prm->cutoff_widths >= 0.0) || !isfinite(prm->cutoff_widths)) return HK_ERR_INVALID;
  if (lines->gamma_self && !(prm->self_fraction >= 0.0 && prm->self_fraction <= 1.0)) return HK_ERR_INVALID;
  const int64_t N = hk_grid_size(nu_min, nu_max, dnu);
  if (N < 1 || N > (1LL << 30)) return HK_ERR_INVALID;
  *N_out = N;
  return HK_OK;
}

// hk_opacity_host: a3 runs as `n` (far, near) launch pairs over consecutive ranges of the grid, from the top down, each pair on
// a stream of its own (streams[i], forked from the call's stream after a1 and joined before the call returns to it) so that
// the CTAs of the next range's far kernel fill the SMs as those of the previous one retire; kappa[lo[i], hi[i]) is final
// once done[i] has passed, and is copied to the host while the later ranges are computed.
constexpr int kMaxChunks = 8;
#ifndef HK_HOST_CHUNKS
#define HK_HOST_CHUNKS 6
#endif
constexpr int kHostChunks = HK_HOST_CHUNKS;
struct GridChunks {
  int64_t align = 0;     // in: > 0 asks for range boundaries at multiples of this many grid points (the k-distribution bin)
  bool aligned = false;  // out: every lo[] / hi[] is such a multiple (or N)
  int n = 1;
  cudaStream_t streams[kMaxChunks] = {};
  cudaEvent_t fork = nullptr;
  cudaEvent_t done[kMaxChunks] = {};
  int64_t lo[kMaxChunks] = {}, hi[kMaxChunks] = {};
};

static int run_opacity(const hk_lines *lines, int64_t n_lines, double T, double P_atm, double q_ratio, double mass_amu,
                       double nu_min, double dnu, double cutoff, int64_t N, double *kappa_out, Scratch &s, const hk_params &prm,
                       cudaStream_t st, double delta_max, GridChunks *chunks = nullptr)
{
  const bool f32 = prm.precision == HK_FP32;
  if (n_lines == 0) {
    if (!prm.accumulate) HK_CUDA(cudaMemsetAsync(kappa_out, 0, (size_t)N * sizeof(double), st));
    if (chunks) {
      chunks->n = 1;
      chunks->lo[0] = 0;
      chunks->hi[0] = N;
      HK_CUDA(cudaEventRecord(chunks->done[0], st));
    }
    return HK_OK;
  }
  const int nb = (int)((N + kPlanBlock - 1) / kPlanBlock);
  int rc = scratch_reserve(s, n_lines, nb, f32, st);
  if (rc != HK_OK) return rc;
  // lines whose window reaches a 256-point span, on average: picks the far kernel's shape
  const double per_span = (double)n_lines * fmin(2.0 * cutoff / dnu + (double)kPlanBlock, (double)N) / (double)N;
  const int shape = f32 ? kShapeF32 : (per_span >= kDenseLinesPerSpan ? kShapeDense : kShapeSparse);
  int grid = 0;
  rc = voigt_grid(shape, &grid);
  if (rc != HK_OK) return rc;
  const int tile = shape == kShapeF32 ? ShF32::TILE : (shape == kShapeDense ? ShDense::TILE : ShSparse::TILE);
  const int n_tiles = (int)((N + tile - 1) / tile);
  if (grid > n_tiles) grid = n_tiles;

  cudaEvent_t *ev = g_ev;
  if (g_timing) {
    for (int i = 0; i < 4; ++i)
      if (!ev[i]) HK_CUDA(cudaEventCreate(&ev[i]));
    HK_CUDA(cudaEventRecord(ev[0], st));
  }
  PrepArgs pa;
  pa.nu0 = lines->nu0; pa.S = lines->S; pa.gamma0 = lines->gamma0; pa.n_T = lines->n_T; pa.E_low = lines->E_low;
  pa.gamma_self = lines->gamma_self; pa.A21 = lines->A21;
  pa.delta = lines->delta; pa.shift_pad = lines->delta ? delta_max * P_atm * (1.0 + 1.0e-12) : 0.0;
  pa.self_fraction = prm.self_fraction; pa.abundance = prm.abundance > 0.0 ? prm.abundance : 1.0;
  pa.cutoff_widths = prm.cutoff_widths;
  pa.n = n_lines;
  pa.T = T; pa.P_atm = P_atm; pa.tfac_half = pow(kT0 / T, 0.5);
  const double m_g = mass_amu * kAmu;
  pa.vth = sqrt(2.0 * kBoltz * T / m_g) / kCLight;
  pa.inv_mg = 1.0 / m_g;
  pa.q_ratio = q_ratio;
  pa.nu_min = nu_min; pa.dnu = dnu; pa.cutoff = cutoff; pa.N = (int)N;
  pa.R2 = f32 ? kR2f : kR2; pa.R3 = f32 ? kR3f : kR3; pa.f32_ladder = f32 ? 1 : 0;
  pa.f32 = f32 ? s.f32 : nullptr;
  pa.ma = s.ma; pa.mb = s.mb; pa.base = s.base; pa.gh2 = s.gh2; pa.core = s.core; pa.near = s.near;
  pa.nb = nb; pa.first_hi = s.first_hi; pa.first_lo = s.first_lo; pa.first_c = s.first_c; pa.queue = s.queue;
  line_prep_kernel<<<(unsigned)((n_lines + 255) / 256), 256, 0, st>>>(pa);
  HK_CUDA(cudaGetLastError());
  if (g_timing) HK_CUDA(cudaEventRecord(ev[1], st));
  VoigtArgs va;
  va.ma = s.ma; va.mb = s.mb; va.base = s.base; va.gh2 = s.gh2; va.core = s.core; va.near = s.near; va.f32 = pa.f32;
  va.dnu_f = (float)dnu;
  va.first_hi = s.first_hi; va.first_lo = s.first_lo; va.first_c = s.first_c; va.queue = s.queue;
  va.nb = nb; va.n_tiles = n_tiles; va.tile0 = 0;
  va.nu_min = nu_min; va.dnu = dnu; va.N = (int)N; va.n_lines = (int)n_lines; va.kappa = kappa_out; va.accumulate = prm.accumulate ? 1 : 0;
  {
    // bound on the 3-ball radius (grid units) of any line that can have grid point j inside its 3-ball:
    // r3 <= s*alpha/dnu with alpha = vth*nu0 and nu0 <= nu_j + r3*dnu, s^2 = max(R3, Gaussian-term radius) (a hair more)
    //   =>  r3 <= s*vth*(nu_min/dnu + j)/(1 - s*vth)
    const double sv = sqrt(fmax(pa.R3, kXgCapSq) + 1.0) * pa.vth;
    if (sv < 0.5) {
      va.r3_slope = sv / (1.0 - sv);
      // (FP32 variant: a line with alpha^2 < 1e-9 sends its whole 1-ball, radius <= 200 alpha < 6.4e-3 cm^-1, to this kernel)
      // (eq. 21: the tables know the unshifted centres, up to shift_pad away from the shifted ones)
      // (and the guard band of f32_guard_points around every centre: three grid points, more on a grid finer than 1.3e-5 cm^-1)
      va.r3_offset = (sv * fmax(nu_min / dnu, 0.0) + (f32 ? f32_guard_points(dnu) + 1.0 + 6.4e-3 / dnu : 4.0) + pa.shift_pad / dnu) /
                     (1.0 - sv);
    } else {  // absurdly hot / light: no useful bound, the near kernel scans every line that touches the span
      va.r3_slope = 0.0;
      va.r3_offset = 4.0e9;
    }
  }
  // ranges only where every one gets a few tiles (a small grid has nothing to overlap)
  const int nch = (chunks && n_tiles >= 8 * chunks->n) ? std::max(1, std::min(chunks->n, kMaxChunks)) : 1;
  const int bpt = tile / kPlanBlock;  // plan blocks per tile
  // hk_opacity_host with a k-table: ranges cut at common multiples of the tile and the bin, so that the bins of a range can be
  // sorted and copied back as soon as that range is final — where the grid holds at least two such units per range
  int64_t unit_tiles = 0, n_units = 0;
  if (chunks && nch > 1 && chunks->align > 0) {
    int64_t g = tile, r = chunks->align;
    while (r) { const int64_t t = g % r; g = r; r = t; }
    const int64_t unit = (int64_t)tile / g * chunks->align;  // lcm, in grid points
    if (N / unit >= 2 * nch) {
      unit_tiles = unit / tile;
      n_units = N / unit;
    }
  }
  if (chunks) chunks->aligned = unit_tiles > 0;
  if (chunks && nch > 1) HK_CUDA(cudaEventRecord(chunks->fork, st));
  for (int c = 0; c < nch; ++c) {     // ranges of whole tiles, from the top of the grid down
    cudaStream_t sc = (chunks && nch > 1) ? chunks->streams[c] : st;
    if (sc != st) HK_CUDA(cudaStreamWaitEvent(sc, chunks->fork, 0));
    // tapered ranges (weights nch + 1 ... 2, top of the grid first): the copy of the last range trails the call, so it is the
    // smallest (measured at config 1: e2e 1.41 ms with the near kernel alone in four parts, 1.22 with six equal (far, near)
    // ranges, 1.21 tapered)
    auto cut = [&](int k) {  // tiles below the k ranges processed last
      const int64_t tot = (int64_t)nch * (nch + 1) / 2 + nch, w = (int64_t)k * (k + 1) / 2 + k;
      if (k >= nch) return n_tiles;
      if (unit_tiles > 0) return (int)((int64_t)n_units * w / tot * unit_tiles);  // whole units of lcm(tile, bin)
      return (int)((int64_t)n_tiles * w / tot);
    };
    const int t_lo = cut(nch - 1 - c), t_hi = cut(nch - c);
    va.tile0 = t_lo;
    va.n_tiles = t_hi - t_lo;
    va.queue = s.queue + c;
    const int g = std::min(grid, va.n_tiles);
    const int b_lo = t_lo * bpt, b_hi = std::min(t_hi * bpt, nb);
    if (g > 0) {  // (a range cut at whole units can be empty)
      if (shape == kShapeF32) voigt_far_kernel<ShF32><<<g, ShF32::WARPS * 32, sizeof(VoigtSmem<ShF32>), sc>>>(va);
      else if (shape == kShapeDense) voigt_far_kernel<ShDense><<<g, ShDense::WARPS * 32, sizeof(VoigtSmem<ShDense>), sc>>>(va);
      else voigt_far_kernel<ShSparse><<<g, ShSparse::WARPS * 32, sizeof(VoigtSmem<ShSparse>), sc>>>(va);
      HK_CUDA(cudaGetLastError());
    }
    if (g_timing && c == nch - 1) HK_CUDA(cudaEventRecord(ev[2], sc));
    va.block0 = b_lo;
    if (b_hi > b_lo) {
      voigt_near_kernel<<<b_hi - b_lo, 32, 0, sc>>>(va);
      HK_CUDA(cudaGetLastError());
    }
    if (chunks) {
      chunks->lo[c] = (int64_t)b_lo * kPlanBlock;
      chunks->hi[c] = std::min<int64_t>((int64_t)b_hi * kPlanBlock, N);
      HK_CUDA(cudaEventRecord(chunks->done[c], sc));
      if (sc != st) HK_CUDA(cudaStreamWaitEvent(st, chunks->done[c], 0));  // join: the call's stream continues after every range
    }
  }
  if (chunks) chunks->n = nch;
  if (g_timing) {
    HK_CUDA(cudaEventRecord(ev[3], st));
    g_ev_pending = true;  // resolved by hk_last_stage_ms(): the call itself stays asynchronous
  }
  return HK_OK;
}

// ------------------------------------------------------------------------------------------------------
// hk_opacity_noalloc (include/hk.h): the work space of a1/a2 as a fixed array in the library image, for callers that may not
// allocate.  Layout: the six record arrays of Scratch at a stride of kNoAllocMaxLines records each, then the FP32 variant's
// records, then (256-byte aligned) first_hi | first_lo | first_c | 16 ticket counters for a grid of kNoAllocMaxBlocks blocks.
// In host code `g_noalloc_scratch` names a host-side shadow of the symbol, NOT device memory: the kernels are given the
// address cudaGetSymbolAddress returns for the current device, looked up once per device.
// ------------------------------------------------------------------------------------------------------
constexpr int64_t kNoAllocMaxLines = HK_NOALLOC_MAX_LINES;
constexpr int64_t kNoAllocMaxPoints = HK_NOALLOC_MAX_POINTS;
constexpr int kNoAllocMaxBlocks = (int)(kNoAllocMaxPoints / kPlanBlock);
constexpr size_t kNoAllocLineBytes = (size_t)kNoAllocMaxLines * (kBytesPerLine + sizeof(LineF32));
constexpr size_t kNoAllocTableBytes = ((((size_t)3 * (kNoAllocMaxBlocks + 1) + 16) * sizeof(int)) + 255) & ~(size_t)255;
constexpr size_t kNoAllocBytes = kNoAllocLineBytes + kNoAllocTableBytes;
static_assert(kNoAllocBytes == (size_t)HK_NOALLOC_SCRATCH_BYTES, "hk.h states the size of the array");
static_assert(kNoAllocMaxPoints % kPlanBlock == 0 && kNoAllocLineBytes % 256 == 0, "table part stays 256-byte aligned");
static __device__ __align__(256) unsigned char g_noalloc_scratch[kNoAllocBytes];

// device address of the array on the current device (first use per device: one cudaGetSymbolAddress, checked)
static int noalloc_scratch(Scratch *out)
{
  static unsigned char *base[64] = {};
  static PerDeviceOnce once;
  int dev = 0;
  HK_CUDA(cudaGetDevice(&dev));
  if (dev < 0 || dev >= 64) return HK_ERR_UNSUPPORTED;
  const int rc = once.run([](int d) {
    void *p = nullptr;
    HK_CUDA(cudaGetSymbolAddress(&p, g_noalloc_scratch));
    if (!p || ((uintptr_t)p & 255u)) return (int)HK_ERR_CUDA;
    base[d] = (unsigned char *)p;
    return (int)HK_OK;
  });
  if (rc != HK_OK) return rc;
  unsigned char *p = base[dev];
  const size_t n = (size_t)kNoAllocMaxLines;
  Scratch s;
  s.ma = (MetaA *)p;
  s.mb = (MetaB *)(p + n * 16);
  s.base = (LineBase *)(p + n * 32);
  s.gh2 = (LineGH2 *)(p + n * 64);
  s.core = (LineCore *)(p + n * 96);
  s.near = (LineNear *)(p + n * 128);
  s.f32 = (LineF32 *)(p + n * kBytesPerLine);
  s.first_hi = (int *)(p + kNoAllocLineBytes);
  s.first_lo = s.first_hi + (kNoAllocMaxBlocks + 1);
  s.first_c = s.first_lo + (kNoAllocMaxBlocks + 1);
  s.queue = s.first_c + (kNoAllocMaxBlocks + 1);
  s.cap_lines = kNoAllocMaxLines;   // scratch_reserve() finds room for every admitted size and allocates nothing
  s.cap_blocks = kNoAllocMaxBlocks;
  *out = s;
  return HK_OK;
}

}  // namespace hk

using namespace hk;

struct hk_ctx {
  hk_lines lines;      // what the kernels read: the caller's arrays, or the library's ordered copy
  void *sorted_buf;    // the ordered copy (NULL when the caller's list was already ascending)
  int64_t n_lines;
  hk_params prm;
  Scratch scratch;
  double delta_max;    // max |delta| of the list (eq. 21), found once at hk_create; 0 without a shift field
};

// max |delta_i| of a device array, on the host (synchronises the stream): sizes the halo of the a2 tables under eq. 21
static int delta_absmax(const double *delta, int64_t n, cudaStream_t st, double *out)
{
  *out = 0.0;
  if (!delta || n <= 0) return HK_OK;
  void *buf = nullptr;
  int rc = pool_alloc(&buf, sizeof(unsigned long long), st);
  if (rc != HK_OK) return rc;
  cudaError_t e = cudaMemsetAsync(buf, 0, sizeof(unsigned long long), st);
  if (e == cudaSuccess) {
    absmax_kernel<<<(unsigned)std::min<int64_t>((n + 255) / 256, 1184), 256, 0, st>>>(delta, n, (unsigned long long *)buf);
    e = cudaGetLastError();
  }
  unsigned long long bits = 0;
  if (e == cudaSuccess) e = cudaMemcpyAsync(&bits, buf, sizeof(bits), cudaMemcpyDeviceToHost, st);
  if (e == cudaSuccess) e = cudaStreamSynchronize(st);
  pool_free(buf, st);
  if (e != cudaSuccess) return cuda_fail(e, "delta_absmax");
  memcpy(out, &bits, sizeof(double));
  if (!isfinite(*out)) return HK_ERR_INVALID;
  return HK_OK;
}

// Resolves the line list the kernels will read: the caller's arrays when they are ascending (promised by lines_sorted = 1,
// or found so by the device check), else an ordered copy (*buf, to be released with pool_free).
static int ordered_lines(const hk_lines *lines, int64_t n_lines, const hk_params *prm, hk_lines *out, void **buf)
{
  *out = *lines;
  *buf = nullptr;
  if (prm->lines_sorted || n_lines < 2) return HK_OK;
  int rc = hk_lines_check_sorted(lines->nu0, n_lines, prm->stream);
  if (rc == HK_OK) return HK_OK;
  if (rc != HK_ERR_UNSORTED) return rc;
  return sort_lines_copy(lines, n_lines, (cudaStream_t)prm->stream, out, buf);
}

extern "C" {

int64_t hk_grid_size(double nu_min, double nu_max, double dnu)
{
  if (!(dnu > 0.0) || !isfinite(nu_min) || !isfinite(nu_max)) return -1;
  const double n = (nu_max - nu_min) / dnu;
  if (!(n < 9.0e18) || !(n > -9.0e18)) return -1;
  return (int64_t)llround(n);
}

static int opacity_impl(const hk_lines *lines, int64_t n_lines, double T, double P_atm, double nu_min, double nu_max,
                        double dnu, double cutoff, double *kappa_out, const hk_params *prm, GridChunks *chunks)
{
  int64_t N = 0;
  int rc = validate(lines, n_lines, T, P_atm, nu_min, nu_max, dnu, cutoff, kappa_out, prm, &N);
  if (rc != HK_OK) return rc;
  cudaStream_t st = (cudaStream_t)prm->stream;
  // eq. 21 needs no copy and no re-ordering: a1 shifts every centre itself and builds its tables from the unshifted, ordered
  // centres with a halo of max |delta| P (found here: one small reduction and a stream synchronisation per one-shot call)
  double dmax = 0.0;
  rc = delta_absmax(lines->delta, n_lines, st, &dmax);
  if (rc != HK_OK) return rc;
  hk_lines use;
  void *sorted_buf = nullptr;
  rc = ordered_lines(lines, n_lines, prm, &use, &sorted_buf);
  if (rc != HK_OK) return rc;
  Scratch s;
  rc = run_opacity(&use, n_lines, T, P_atm, prm->q_ratio, prm->mass_amu, nu_min, dnu, cutoff, N, kappa_out, s, *prm, st, dmax,
                   chunks);
  scratch_release(s, st);
  pool_free(sorted_buf, st);
  return rc;
}

int hk_opacity(const hk_lines *lines, int64_t n_lines, double T, double P_atm, double nu_min, double nu_max, double dnu,
               double cutoff, double *kappa_out, const hk_params *prm)
{
  return opacity_impl(lines, n_lines, T, P_atm, nu_min, nu_max, dnu, cutoff, kappa_out, prm, nullptr);
}

// hk_opacity on the fixed work space (see include/hk.h): no allocation, no host wait
int hk_opacity_noalloc(const hk_lines *lines, int64_t n_lines, double T, double P_atm, double nu_min, double nu_max,
                       double dnu, double cutoff, double *kappa_out, const hk_params *prm)
{
  int64_t N = 0;
  int rc = validate(lines, n_lines, T, P_atm, nu_min, nu_max, dnu, cutoff, kappa_out, prm, &N);
  if (rc != HK_OK) return rc;
  if (n_lines > kNoAllocMaxLines) {
    snprintf(g_cuda_err, sizeof(g_cuda_err),
             "hk_opacity_noalloc: %lld lines, the fixed work space holds HK_NOALLOC_MAX_LINES = %lld (feed the list in ordered "
             "pieces with accumulate = 1, or call hk_opacity)", (long long)n_lines, (long long)kNoAllocMaxLines);
    return HK_ERR_UNSUPPORTED;
  }
  if (N > kNoAllocMaxPoints) {
    snprintf(g_cuda_err, sizeof(g_cuda_err),
             "hk_opacity_noalloc: %lld grid points, the fixed work space serves HK_NOALLOC_MAX_POINTS = %lld (split the grid "
             "into ranges, or call hk_opacity)", (long long)N, (long long)kNoAllocMaxPoints);
    return HK_ERR_UNSUPPORTED;
  }
  if (!prm->lines_sorted) {
    snprintf(g_cuda_err, sizeof(g_cuda_err),
             "hk_opacity_noalloc: lines_sorted must be 1 (checking or re-ordering the list needs an allocation and a host wait)");
    return HK_ERR_UNSUPPORTED;
  }
  if (lines->delta) {
    snprintf(g_cuda_err, sizeof(g_cuda_err),
             "hk_opacity_noalloc: a pressure-shift field (delta) is not served (its halo needs a reduction and a host wait)");
    return HK_ERR_UNSUPPORTED;
  }
  Scratch s;
  rc = noalloc_scratch(&s);
  if (rc != HK_OK) return rc;
  const int timing = g_timing;  // the stage events of hk_set_timing are created on demand: not on this path
  g_timing = 0;
  rc = run_opacity(lines, n_lines, T, P_atm, prm->q_ratio, prm->mass_amu, nu_min, dnu, cutoff, N, kappa_out, s, *prm,
                   (cudaStream_t)prm->stream, 0.0);
  g_timing = timing;
  return rc;  // nothing to release: `s` only points into the array
}

// copy stream and events of hk_opacity_host, one set per host thread (re-made when the thread changes device)
struct HostCopy {
  int dev = -1;
  cudaStream_t copy = nullptr;
  cudaStream_t range[kMaxChunks] = {};  // one per grid range, earlier ranges at higher priority
  cudaEvent_t fork = nullptr;
  cudaEvent_t done[kMaxChunks] = {};
  cudaEvent_t sorted[kMaxChunks] = {};  // the k-distribution of a range's bins is done
  cudaEvent_t copied = nullptr;
};
static thread_local HostCopy g_hc;
static int host_copy_get(HostCopy **out)
{
  int dev = 0;
  HK_CUDA(cudaGetDevice(&dev));
  HostCopy &h = g_hc;
  if (h.dev != dev) {
    h = HostCopy();  // a set made on another device is abandoned (a thread that hops devices is not the case served)
    HK_CUDA(cudaStreamCreateWithFlags(&h.copy, cudaStreamNonBlocking));
    for (int i = 0; i < kMaxChunks; ++i) HK_CUDA(cudaEventCreateWithFlags(&h.done[i], cudaEventDisableTiming));
    for (int i = 0; i < kMaxChunks; ++i) HK_CUDA(cudaEventCreateWithFlags(&h.sorted[i], cudaEventDisableTiming));
    HK_CUDA(cudaEventCreateWithFlags(&h.fork, cudaEventDisableTiming));
    int prio_lo = 0, prio_hi = 0;  // numerically lower = higher priority
    HK_CUDA(cudaDeviceGetStreamPriorityRange(&prio_lo, &prio_hi));
    for (int i = 0; i < kMaxChunks; ++i)
      HK_CUDA(cudaStreamCreateWithPriority(&h.range[i], cudaStreamNonBlocking, std::min(prio_lo, prio_hi + i)));
    HK_CUDA(cudaEventCreateWithFlags(&h.copied, cudaEventDisableTiming));
    h.dev = dev;
  }
  *out = &h;
  return HK_OK;
}

int hk_opacity_host(const hk_lines *lines_host, int64_t n_lines, double T, double P_atm, double nu_min, double nu_max,
                    double dnu, double cutoff, double *kappa_host_out, double bin_width, int n_g, double *k_host_out,
                    const hk_params *prm)
{
  if (!lines_host || !prm || n_lines < 0 || (!kappa_host_out && !k_host_out)) return HK_ERR_INVALID;
  if (prm->accumulate && !kappa_host_out) return HK_ERR_INVALID;  // the running sum of a mixture is read from it
  if (n_lines > 0 && (!lines_host->nu0 || !lines_host->S || !lines_host->gamma0)) return HK_ERR_INVALID;
  const int64_t N = hk_grid_size(nu_min, nu_max, dnu);
  if (N < 1 || N > (1LL << 30)) return HK_ERR_INVALID;
  int64_t n_bins = 0;
  if (k_host_out) {
    if (!pos_finite(bin_width) || n_g < 1 || n_g > 128) return HK_ERR_INVALID;
    const double ppb_d = nearbyint(bin_width / dnu);
    if (ppb_d < 1.0 || fmod((double)N, ppb_d) != 0.0) return HK_ERR_INVALID;
    n_bins = N / (int64_t)ppb_d;
  }
  cudaStream_t st = (cudaStream_t)prm->stream;
  HostCopy *hc = nullptr;
  {
    int rch = host_copy_get(&hc);
    if (rch != HK_OK) return rch;
  }
  constexpr int NF = 8;
  const double *src[NF] = {lines_host->nu0, lines_host->S, lines_host->gamma0, lines_host->n_T, lines_host->E_low,
                           lines_host->gamma_self, lines_host->A21, lines_host->delta};
  const size_t fbytes = ((size_t)n_lines * sizeof(double) + 255) & ~(size_t)255;
  const size_t kappa_bytes = ((size_t)N * sizeof(double) + 255) & ~(size_t)255;
  void *dev = nullptr;
  int rc = pool_alloc(&dev, NF * fbytes + kappa_bytes + (size_t)n_bins * n_g * sizeof(double), st);
  if (rc != HK_OK) return rc;
  const double *dptr[NF] = {};
  cudaError_t e = cudaSuccess;
  for (int f = 0; f < NF && e == cudaSuccess; ++f) {
    if (!src[f] || n_lines == 0) continue;
    double *d = (double *)((char *)dev + f * fbytes);
    e = cudaMemcpyAsync(d, src[f], (size_t)n_lines * sizeof(double), cudaMemcpyHostToDevice, st);
    dptr[f] = d;
  }
  double *d_kappa = (double *)((char *)dev + NF * fbytes);
  double *d_k = (double *)((char *)dev + NF * fbytes + kappa_bytes);
  if (e == cudaSuccess && prm->accumulate && kappa_host_out)  // a mixture's running sum lives in the caller's host buffer
    e = cudaMemcpyAsync(d_kappa, kappa_host_out, (size_t)N * sizeof(double), cudaMemcpyHostToDevice, st);
  if (e == cudaSuccess) {
    hk_lines dl = {dptr[0], dptr[1], dptr[2], dptr[3], dptr[4], dptr[5], dptr[6], dptr[7]};
    // kappa goes back range by range on a second stream while the near kernel still works on the later ranges: the
    // device -> host copy of 8 B/point is a quarter of the call at config 1
    GridChunks ch;
    ch.n = kappa_host_out ? kHostChunks : 1;
    // Sorting the bins range by range (ranges cut at common multiples of tile and bin, each range's k-distribution on its own
    // stream, rows copied behind kappa) is built and tested but OFF: at config 1 it measured 1.25 ms per call against 1.20 ms
    // with the k-distribution taken once after the last range (profiles/r03_README.md); -DHK_HOST_KDIST_BY_RANGE turns it on.
#ifdef HK_HOST_KDIST_BY_RANGE
    ch.align = (kappa_host_out && k_host_out) ? N / n_bins : 0;  // points per bin
#endif
    ch.fork = hc->fork;
    for (int i = 0; i < kMaxChunks; ++i) ch.streams[i] = hc->range[i];
    bool copies_pending = false;
    for (int i = 0; i < kMaxChunks; ++i) ch.done[i] = hc->done[i];
    rc = opacity_impl(&dl, n_lines, T, P_atm, nu_min, nu_max, dnu, cutoff, d_kappa, prm, &ch);
    // ranges cut at bin boundaries (ch.aligned): the bins of each range are sorted on the range's own stream right behind its
    // near kernel, and their k-table rows follow the range's kappa to the host — nothing is left to do after the last range
    const bool k_by_range = rc == HK_OK && kappa_host_out && k_host_out && ch.aligned && ch.n > 1;
    if (k_by_range) {
      const int64_t ppb = N / n_bins;
      for (int c = 0; c < ch.n && rc == HK_OK && e == cudaSuccess; ++c) {
        if (ch.hi[c] <= ch.lo[c]) continue;
        rc = hk_kdist(d_kappa + ch.lo[c], ch.hi[c] - ch.lo[c], dnu, bin_width, n_g, d_k + ch.lo[c] / ppb * n_g, ch.streams[c]);
        if (rc == HK_OK) e = cudaEventRecord(hc->sorted[c], ch.streams[c]);
      }
    }
    if (rc == HK_OK && kappa_host_out) {
      for (int c = 0; c < ch.n && e == cudaSuccess; ++c) {
        e = cudaStreamWaitEvent(hc->copy, ch.done[c], 0);
        if (e == cudaSuccess && ch.hi[c] > ch.lo[c])
          e = cudaMemcpyAsync(kappa_host_out + ch.lo[c], d_kappa + ch.lo[c], (size_t)(ch.hi[c] - ch.lo[c]) * sizeof(double),
                              cudaMemcpyDeviceToHost, hc->copy);
      }
      // the k-table rows behind all of kappa (a few hundred KB): a sort that waits for free SMs must not hold up the big copies
      for (int c = 0; k_by_range && c < ch.n && e == cudaSuccess; ++c) {
        if (ch.hi[c] <= ch.lo[c]) continue;
        const int64_t ppb = N / n_bins, b0 = ch.lo[c] / ppb, nb_c = (ch.hi[c] - ch.lo[c]) / ppb;
        e = cudaStreamWaitEvent(hc->copy, hc->sorted[c], 0);
        if (e == cudaSuccess)
          e = cudaMemcpyAsync(k_host_out + b0 * n_g, d_k + b0 * n_g, (size_t)nb_c * n_g * sizeof(double), cudaMemcpyDeviceToHost,
                              hc->copy);
      }
      if (e == cudaSuccess) e = cudaEventRecord(hc->copied, hc->copy);
      copies_pending = e == cudaSuccess;
    }
    if (!k_by_range) {
      if (rc == HK_OK && e == cudaSuccess && k_host_out) rc = hk_kdist(d_kappa, N, dnu, bin_width, n_g, d_k, prm->stream);
      if (rc == HK_OK && e == cudaSuccess && k_host_out)
        e = cudaMemcpyAsync(k_host_out, d_k, (size_t)n_bins * n_g * sizeof(double), cudaMemcpyDeviceToHost, st);
    }
    if (copies_pending && e == cudaSuccess) e = cudaStreamWaitEvent(st, hc->copied, 0);  // st frees the buffer after them
  }
  if (e != cudaSuccess || rc != HK_OK) {  // error path: nothing may still read the buffer
    cudaStreamSynchronize(hc->copy);
    for (int i = 0; i < kMaxChunks; ++i) cudaStreamSynchronize(hc->range[i]);
  }
  pool_free(dev, st);
  const cudaError_t es = cudaStreamSynchronize(st);
  if (rc != HK_OK) return rc;
  if (e != cudaSuccess) return cuda_fail(e, "hk_opacity_host copy");
  if (es != cudaSuccess) return cuda_fail(es, "hk_opacity_host synchronize");
  return HK_OK;
}

int hk_create(const hk_lines *lines, int64_t n_lines, const hk_params *prm, hk_ctx **out)
{
  if (!lines || !prm || !out || n_lines < 0) return HK_ERR_INVALID;
  if (n_lines > 0 && (!lines->nu0 || !lines->S || !lines->gamma0)) return HK_ERR_INVALID;
  if (n_lines > 2000000000LL) return HK_ERR_UNSUPPORTED;
  if (!pos_finite(prm->mass_amu)) return HK_ERR_INVALID;
  if (prm->precision != HK_FP64 && prm->precision != HK_FP32) return HK_ERR_INVALID;
  hk_ctx *c = new (std::nothrow) hk_ctx();
  if (!c) return HK_ERR_NOMEM;
  c->n_lines = n_lines;
  c->prm = *prm;
  int rc = ordered_lines(lines, n_lines, prm, &c->lines, &c->sorted_buf);
  if (rc != HK_OK) {
    delete c;
    return rc;
  }
  c->prm.lines_sorted = 1;
  rc = delta_absmax(c->lines.delta, n_lines, (cudaStream_t)prm->stream, &c->delta_max);  // eq. 21: halo of the a2 tables
  if (rc != HK_OK) {
    pool_free(c->sorted_buf, (cudaStream_t)prm->stream);
    delete c;
    return rc;
  }
  *out = c;
  return HK_OK;
}

int hk_opacity_ctx(hk_ctx *ctx, double T, double P_atm, double q_ratio, double nu_min, double nu_max, double dnu,
                   double cutoff, double *kappa_out)
{
  if (!ctx) return HK_ERR_INVALID;
  hk_params p = ctx->prm;
  p.q_ratio = q_ratio;
  int64_t N = 0;
  int rc = validate(&ctx->lines, ctx->n_lines, T, P_atm, nu_min, nu_max, dnu, cutoff, kappa_out, &p, &N);
  if (rc != HK_OK) return rc;
  return run_opacity(&ctx->lines, ctx->n_lines, T, P_atm, q_ratio, p.mass_amu, nu_min, dnu, cutoff, N, kappa_out,
                     ctx->scratch, p, (cudaStream_t)p.stream, ctx->delta_max);
}

int hk_destroy(hk_ctx *ctx)
{
  if (!ctx) return HK_ERR_INVALID;
  cudaStream_t st = (cudaStream_t)ctx->prm.stream;
  scratch_release(ctx->scratch, st);
  pool_free(ctx->sorted_buf, st);
  cudaStreamSynchronize(st);
  delete ctx;
  return HK_OK;
}

int hk_lines_check_sorted(const double *nu0_device, int64_t n_lines, void *stream)
{
  if (n_lines < 0 || (n_lines > 0 && !nu0_device)) return HK_ERR_INVALID;
  if (n_lines < 2) return HK_OK;
  cudaStream_t st = (cudaStream_t)stream;
  int *flag = nullptr;
  { void *pf = nullptr; int rcp = pool_alloc(&pf, sizeof(int), st); if (rcp != HK_OK) return rcp; flag = (int *)pf; }
  HK_CUDA(cudaMemsetAsync(flag, 0, sizeof(int), st));
  check_sorted_kernel<<<(unsigned)((n_lines + 255) / 256), 256, 0, st>>>(nu0_device, n_lines, flag);
  int h = 0;
  cudaError_t e = cudaMemcpyAsync(&h, flag, sizeof(int), cudaMemcpyDeviceToHost, st);
  if (e == cudaSuccess) e = cudaStreamSynchronize(st);
  cudaFreeAsync(flag, st);
  if (e != cudaSuccess) return cuda_fail(e, "check_sorted");
  return h ? HK_ERR_UNSORTED : HK_OK;
}

int64_t hk_count_evals(const double *nu0_host, int64_t n_lines, double nu_min, int64_t N, double dnu, double cutoff)
{
  if (!nu0_host || n_lines < 0 || N < 1 || !(dnu > 0.0) || !(cutoff > 0.0)) return -1;
  int64_t total = 0;
  for (int64_t i = 0; i < n_lines; ++i) {
    double lo = ceil(((nu0_host[i] - cutoff) - nu_min) / dnu);
    double hi = floor(((nu0_host[i] + cutoff) - nu_min) / dnu);
    if (!(lo > 0.0)) lo = 0.0;
    if (!(hi < (double)(N - 1))) hi = (double)(N - 1);
    if (hi >= lo) total += (int64_t)hi - (int64_t)lo + 1;
  }
  return total;
}

int hk_regime_census(const double *nu0_host, const double *gamma0_host, int64_t n_lines, double T, double P_atm,
                     double mass_amu, double nu_min, int64_t N, double dnu, double cutoff, int precision,
                     int64_t counts_out[5])
{
  if (precision != HK_FP64 && precision != HK_FP32) return HK_ERR_INVALID;
  const double R2 = precision == HK_FP32 ? kR2f : kR2, R3 = precision == HK_FP32 ? kR3f : kR3;
  if (!nu0_host || !gamma0_host || !counts_out || n_lines < 0 || N < 1 || !pos_finite(T) || !pos_finite(P_atm) ||
      !pos_finite(mass_amu) || !pos_finite(dnu) || !pos_finite(cutoff))
    return HK_ERR_INVALID;
  const double vth = sqrt(2.0 * kBoltz * T / (mass_amu * kAmu)) / kCLight;
  const double tfac = pow(kT0 / T, 0.5);
  // points of the window [lo, hi] with |nu_j - nu0| < rho  (rho in cm^-1)
  auto within = [&](double nu0, double rho, int64_t lo, int64_t hi) -> int64_t {
    if (!(rho > 0.0)) return 0;
    double a = ceil(((nu0 - rho) - nu_min) / dnu), b = floor(((nu0 + rho) - nu_min) / dnu);
    if (a * dnu + nu_min <= nu0 - rho) a += 1.0;  // strict inequality at the edges
    if (b * dnu + nu_min >= nu0 + rho) b -= 1.0;
    const int64_t ia = a < (double)lo ? lo : (int64_t)a, ib = b > (double)hi ? hi : (int64_t)b;
    return ib >= ia ? ib - ia + 1 : 0;
  };
  int64_t c[5] = {0, 0, 0, 0, 0};
  for (int64_t i = 0; i < n_lines; ++i) {
    const double nu0 = nu0_host[i];
    double lo = ceil(((nu0 - cutoff) - nu_min) / dnu), hi = floor(((nu0 + cutoff) - nu_min) / dnu);
    if (!(lo > 0.0)) lo = 0.0;
    if (!(hi < (double)(N - 1))) hi = (double)(N - 1);
    if (hi < lo) continue;
    const int64_t jl = (int64_t)lo, jh = (int64_t)hi, tot = jh - jl + 1;
    double alpha = nu0 * vth;
    if (!(alpha > 0.0)) { c[0] += tot; continue; }
    const double gamma = gamma0_host[i] * P_atm * tfac, a2 = alpha * alpha, g2 = gamma * gamma, y = gamma / alpha;
    auto rho = [&](double R) { const double t = R * a2 - g2; return t > 0.0 ? sqrt(t) : 0.0; };
    const double xc2 = core_xc2(y);
    const double R1 = r1_sq(y, precision == HK_FP32);
    const int64_t n2 = within(nu0, rho(R2), jl, jh), n3 = within(nu0, rho(R3), jl, jh);
    const int64_t n1 = std::max(within(nu0, rho(R1), jl, jh), n2);  // the 2-point rule fills [R2, R1) when R1 > R2
    const int64_t nc = xc2 > 0.0 ? within(nu0, sqrt(xc2) * alpha, jl, jh) : 0;
    const int64_t ncore = nc < n3 ? nc : n3;
    c[0] += tot - n1; c[1] += n1 - n2; c[2] += n2 - n3; c[3] += n3 - ncore; c[4] += ncore;
  }
  for (int k = 0; k < 5; ++k) counts_out[k] = c[k];
  return HK_OK;
}

int hk_gauss_legendre(int n_g, double *g, double *w)
{
  if (n_g < 1 || n_g > 4096 || !g || !w) return HK_ERR_INVALID;
  // roots of P_n on (-1,1) by Newton from the asymptotic guess, symmetric pairs; mapped to (0,1)
  const long double pi = 3.14159265358979323846264338327950288L;
  const int half = (n_g + 1) / 2;
  for (int i = 0; i < half; ++i) {
    long double z = cosl(pi * (i + 0.75L) / (n_g + 0.5L));
    long double dp = 1.0L;
    for (int it = 0; it < 64; ++it) {
      long double pm = 1.0L, pc = z;  // P_0, P_1
      for (int k = 2; k <= n_g; ++k) {
        const long double pn = ((2 * k - 1) * z * pc - (k - 1) * pm) / k;
        pm = pc; pc = pn;
      }
      if (n_g == 1) { pm = 1.0L; pc = z; }
      dp = n_g * (z * pc - pm) / (z * z - 1.0L);
      const long double dz = pc / dp;
      z -= dz;
      if (fabsl(dz) < 1e-19L) {
        long double qm = 1.0L, qc = z;
        for (int k = 2; k <= n_g; ++k) {
          const long double qn = ((2 * k - 1) * z * qc - (k - 1) * qm) / k;
          qm = qc; qc = qn;
        }
        dp = n_g * (z * qc - qm) / (z * z - 1.0L);
        break;
      }
    }
    const long double wt = 1.0L / ((1.0L - z * z) * dp * dp);  // half of 2/((1-z^2) P'^2): weights on (0,1)
    g[n_g - 1 - i] = (double)(0.5L * (1.0L + z));
    g[i] = (double)(0.5L * (1.0L - z));
    w[n_g - 1 - i] = (double)wt;
    w[i] = (double)wt;
  }
  return HK_OK;
}

int hk_voigt_K(const double *x, const double *y, int64_t n, double *out, int precision, void *stream)
{
  if (n < 0 || (n > 0 && (!x || !y || !out))) return HK_ERR_INVALID;
  if (precision != HK_FP64 && precision != HK_FP32) return HK_ERR_INVALID;
  if (n == 0) return HK_OK;
  if (precision == HK_FP32) voigt_K_kernel<true><<<(unsigned)((n + 127) / 128), 128, 0, (cudaStream_t)stream>>>(x, y, n, out);
  else voigt_K_kernel<false><<<(unsigned)((n + 127) / 128), 128, 0, (cudaStream_t)stream>>>(x, y, n, out);
  HK_CUDA(cudaGetLastError());
  return HK_OK;
}

int hk_fp64_peak(double *inst_per_s_out, void *stream)
{
  if (!inst_per_s_out) return HK_ERR_INVALID;
  cudaStream_t st = (cudaStream_t)stream;
  int dev = 0, sms = 0;
  HK_CUDA(cudaGetDevice(&dev));
  HK_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  double *buf = nullptr;
  { void *pb = nullptr; int rcp = pool_alloc(&pb, 64, st); if (rcp != HK_OK) return rcp; buf = (double *)pb; }
  cudaEvent_t e0, e1;
  HK_CUDA(cudaEventCreate(&e0));
  HK_CUDA(cudaEventCreate(&e1));
  const int iters = 20000, grid = sms * 4, thr = 256;
  float best = 1e30f;
  for (int r = 0; r < 4; ++r) {
    HK_CUDA(cudaEventRecord(e0, st));
    dfma_peak_kernel<<<grid, thr, 0, st>>>(buf, iters, 1.0000001, 1e-9);
    HK_CUDA(cudaEventRecord(e1, st));
    HK_CUDA(cudaEventSynchronize(e1));
    float ms = 0.f;
    HK_CUDA(cudaEventElapsedTime(&ms, e0, e1));
    if (r > 0 && ms < best) best = ms;
  }
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  cudaFreeAsync(buf, st);
  *inst_per_s_out = (double)grid * thr * (double)iters * 8.0 / (best * 1e-3);
  return HK_OK;
}

int hk_fp32_peak(double *inst_per_s_out, void *stream)
{
  if (!inst_per_s_out) return HK_ERR_INVALID;
  cudaStream_t st = (cudaStream_t)stream;
  int dev = 0, sms = 0;
  HK_CUDA(cudaGetDevice(&dev));
  HK_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  float *buf = nullptr;
  { void *pb = nullptr; int rcp = pool_alloc(&pb, 64, st); if (rcp != HK_OK) return rcp; buf = (float *)pb; }
  cudaEvent_t e0, e1;
  HK_CUDA(cudaEventCreate(&e0));
  HK_CUDA(cudaEventCreate(&e1));
  const int iters = 20000, grid = sms * 8, thr = 256;
  float best = 1e30f;
  for (int r = 0; r < 4; ++r) {
    HK_CUDA(cudaEventRecord(e0, st));
    ffma_peak_kernel<<<grid, thr, 0, st>>>(buf, iters, 1.0000001f, 1e-9f);
    HK_CUDA(cudaEventRecord(e1, st));
    HK_CUDA(cudaEventSynchronize(e1));
    float ms = 0.f;
    HK_CUDA(cudaEventElapsedTime(&ms, e0, e1));
    if (r > 0 && ms < best) best = ms;
  }
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  cudaFreeAsync(buf, st);
  *inst_per_s_out = (double)grid * thr * (double)iters * 16.0 / (best * 1e-3);
  return HK_OK;
}

int hk_set_timing(int on)
{
  g_timing = on ? 1 : 0;
  return HK_OK;
}

int hk_last_stage_ms(float ms_out[3])
{
  if (!ms_out) return HK_ERR_INVALID;
  if (g_ev_pending) {
    HK_CUDA(cudaEventSynchronize(g_ev[3]));
    for (int i = 0; i < 3; ++i) HK_CUDA(cudaEventElapsedTime(&g_stage_ms[i], g_ev[i], g_ev[i + 1]));
    g_ev_pending = false;
  }
  for (int i = 0; i < 3; ++i) ms_out[i] = g_stage_ms[i];
  return HK_OK;
}

int hk_trim(void)
{
  cudaMemPool_t mp = nullptr;
  int rc = lib_pool(&mp);
  if (rc != HK_OK) return rc;
  HK_CUDA(cudaDeviceSynchronize());
  HK_CUDA(cudaMemPoolTrimTo(mp, 0));
  return HK_OK;
}

const char *hk_strerror(int code)
{
  switch (code) {
    case HK_OK: return "ok";
    case HK_ERR_INVALID: return "invalid argument";
    case HK_ERR_CUDA: return "CUDA runtime error";
    case HK_ERR_NOMEM: return "out of memory";
    case HK_ERR_UNSORTED: return "line centres are not ascending";
    case HK_ERR_UNSUPPORTED: return "unsupported request";
    default: return "unknown error";
  }
}

const char *hk_last_cuda_error(void) { return g_cuda_err; }
#ifdef HK_DEBUG_CHECKS
const char *hk_version(void) { return "hk 0.1 (sm_100a, checked: HK_DEBUG_CHECKS)"; }
#else
const char *hk_version(void) { return "hk 0.1 (sm_100a)"; }
#endif

}  // extern "C"
