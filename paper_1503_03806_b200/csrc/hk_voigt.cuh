// hk_voigt.cuh — device Voigt-profile arithmetic for sm_100a (FP64 pipe; no tensor cores: not a contraction).
//
// The profile value of one line at one grid point (eq. 19),
//     V(d) = K(d/alpha, gamma/alpha) / (alpha sqrt(pi)),     K(x,y) = H_V = Re w(x+iy)
// is evaluated in one of five regimes chosen on r^2 = x^2 + y^2 (PAPER.md:197 gives the three-regime
// structure and calls its switch points "trial-and-error"; DESIGN.md "Regimes" derives these):
//
//   r^2 >= 6.0e6 : 1-point Gauss-Hermite  (a Lorentzian)                      5 FP64 + 1 MUFU per point
//   r^2 >= 3200  : 2-point Gauss-Hermite                                       7 FP64 + 1 MUFU
//   r^2 >= 280   : 3-point Gauss-Hermite ("third-order", Letchworth & Benner) 11 FP64 + 1 MUFU
//   r^2 >= 44    : 6-point Gauss-Hermite                                      19 FP64 + 3 MUFU
//   else         : Algorithm-916-type series (Zaghloul & Ali 2012), step a = 0.7, ~16 terms
//
// n-point Gauss-Hermite in dimensional form (no 1/alpha, safe as alpha -> 0), with nodes +-t_k, normalised
// weights wn_k (sum 1) and q = d^2:
//     V = (gamma/pi) sum_k wn_k / ((d - t_k alpha)^2 + gamma^2)
// a +-t pair collapses to one rational:   2 wn (E + 2 t^2 alpha^2) / (E^2 + f),
//     E = q + (gamma^2 - t^2 alpha^2),   f = 4 t^2 alpha^2 gamma^2.
// Division = MUFU.RCP64H seed (2^-20) + one Newton step (2^-40); the 1e-6 parity bar needs no more.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace hk {

constexpr double kR1 = 6.0e6;   // 1-point rule from here   (max rel. error 2.5e-7 on the ring)
constexpr double kR2 = 3200.0;  // 2-point rule             (2.4e-7)
constexpr double kR3 = 280.0;   // 3-point rule             (2.4e-7)
constexpr double kRc = 44.0;    // 6-point rule from here (3.7e-8); series below
constexpr double kXcapSq = 289.0;  // series usable up to x = 17 (32 lane-held terms at a = 0.7)

constexpr double kPi = 3.14159265358979323846;
constexpr double kSqrtPi = 1.772453850905516027298167;
constexpr double kInvSqrtPi = 0.5641895835477562869480795;

// Algorithm-916-type series constants, step a = 0.7 (truncation error 1.1e-8 relative, uniform in y)
constexpr double kA = 0.7;
constexpr double kExpA2 = 0.61262639418441606898858;      // exp(-a^2)
constexpr double kExp2A2 = 0.3753110988513995387142672;   // exp(-2 a^2)
constexpr double k2AoverPi = 0.4456338406573069401528745; // 2a/pi
constexpr double kAoverPi = 0.2228169203286534700764373;  // a/pi

// 6-point Gauss-Hermite: t_k^2 and normalised weights w_k/sqrt(pi) of the three +- pairs
constexpr double kT6sq0 = 0.1901635091934881328718554, kW6_0 = 0.4088284695560292260885378;
constexpr double kT6sq1 = 1.784492748543251591186722, kW6_1 = 0.08861574604191452748085588;
constexpr double kT6sq2 = 5.525343742263260275941422, kW6_2 = 0.002555784402056246430606291;

constexpr unsigned kFull = 0xffffffffu;

__device__ __forceinline__ double rcp_seed(double x)
{
  double r;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
  return r;
}
// 1/x to ~2^-40: one Newton step on the 2^-20 seed (2 DFMA + 1 MUFU)
__device__ __forceinline__ double rcp_nr(double x)
{
  double r0 = rcp_seed(x);
  double e = fma(-x, r0, 1.0);
  return fma(r0, e, r0);
}

// ---- wing rules: contribution amp * V(d) added to acc --------------------------------------------------
// 1-point: A1/(d^2+g2), A1 = amp*gamma/pi
__device__ __forceinline__ double gh1_acc(double acc, double d, double A1, double g2)
{
  double D = fma(d, d, g2);
  return fma(A1, rcp_nr(D), acc);
}
// 2-point (t^2 = 1/2, wn = 1/2): A1 (E + alpha^2)/(E^2 + f2), E = d^2 + e2, e2 = g2 - a2/2, f2 = 2 a2 g2
__device__ __forceinline__ double gh2_acc(double acc, double d, double A1, double e2, double f2, double A1a2)
{
  double E = fma(d, d, e2);
  double D = fma(E, E, f2);
  double B = fma(A1, E, A1a2);
  return fma(B, rcp_nr(D), acc);
}
// 3-point (t = 0 with wn = 2/3; t^2 = 3/2 with wn = 1/6): A1 [ (2/3)/R + (1/3)(E + 3 a2)/(E^2 + f3) ]
//   R = d^2 + g2, E = d^2 + e3, e3 = g2 - 1.5 a2, f3 = 6 a2 g2; c0 = 2 A1/3, c3 = A1/3, c3a = A1 a2
__device__ __forceinline__ double gh3_acc(double acc, double d, double g2, double e3, double f3, double c0, double c3,
                                          double c3a)
{
  double R = fma(d, d, g2);
  double E = fma(d, d, e3);
  double D = fma(E, E, f3);
  double B = fma(c3, E, c3a);
  double num = fma(c0, D, B * R);
  return fma(num, rcp_nr(R * D), acc);
}
// one +-t pair of an n-point rule: 2 wn (E + 2 t^2 a2)/(E^2 + f)
__device__ __forceinline__ double gh_pair(double q, double g2, double a2, double tsq, double wn)
{
  double E = q + (g2 - tsq * a2);
  double D = fma(E, E, 4.0 * tsq * a2 * g2);
  return 2.0 * wn * (E + 2.0 * tsq * a2) * rcp_nr(D);
}
// 6-point: V/(gamma/pi)
__device__ __forceinline__ double gh6_shape(double q, double g2, double a2)
{
  return gh_pair(q, g2, a2, kT6sq0, kW6_0) + gh_pair(q, g2, a2, kT6sq1, kW6_1) + gh_pair(q, g2, a2, kT6sq2, kW6_2);
}

// ---- core: Algorithm-916-type series (restated in DESIGN.md "Core series") ----------------
//   K(x,y) = exp(-x^2) [ erfcx(y) cos(2xy) + (2a/pi) sin^2(xy)/y - (2a/pi) y cos(2xy) S1(y) ]
//          + (a/pi) y sum_{n>=1} [exp(-(an-x)^2) + exp(-(an+x)^2)] / (a^2 n^2 + y^2),
//   S1(y) = sum_{n>=1} exp(-a^2 n^2)/(a^2 n^2 + y^2).
// y is a per-line constant, so the warp holds 1/(a^2 n^2 + y^2) for n = lane+1 in a register and the series
// loop broadcasts it with SHFL; exp(-(an -+ x)^2) advance by the recurrence
//   T(n) = T(n-1) * exp(-a^2 (2n-1)) * exp(+-2 a x),  T(0) = exp(-x^2)   (each T <= 1: no overflow).
struct CoreLine {
  double y, erfcx_y, S1, wn;  // wn is lane-dependent: 1/(a^2 (lane+1)^2 + y^2)
  int nterms;
};

// All 32 lanes must call (warp-collective).
__device__ __forceinline__ CoreLine core_setup(double y, double xmax)
{
  CoreLine c;
  const int lane = threadIdx.x & 31;
  const double n = (double)(lane + 1);
  const double an2 = kA * kA * n * n;
  c.y = y;
  c.wn = 1.0 / (an2 + y * y);
  double term = exp(-an2) * c.wn;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) term += __shfl_xor_sync(kFull, term, o);
  c.S1 = term;
  c.erfcx_y = erfcx(y);
  int nt = (int)ceil((xmax + 4.4) / kA);
  c.nterms = nt > 32 ? 32 : nt;
  return c;
}

// All 32 lanes must call with the same CoreLine (warp-collective: SHFL inside).  x >= 0, x <= 17.
__device__ __forceinline__ double core_K(double x, const CoreLine &c)
{
  const double ex2 = exp(-x * x);
  const double p = exp(2.0 * kA * x);
  const double qq = 1.0 / p;
  const double s = sin(x * c.y);
  const double s2 = s * s;
  const double c2 = fma(-2.0, s2, 1.0);
  double Tm = ex2, Tp = ex2, ck = kExpA2, sum = 0.0;
  for (int k = 0; k < c.nterms; ++k) {
    Tm *= ck * p;
    Tp *= ck * qq;
    const double w = __shfl_sync(kFull, c.wn, k);
    sum = fma(w, Tm + Tp, sum);
    ck *= kExp2A2;
  }
  const double head = c.erfcx_y * c2 + k2AoverPi * (s * (s / c.y)) - k2AoverPi * c.y * c2 * c.S1;
  return fma(ex2, head, kAoverPi * c.y * sum);
}

// Per-line quantities the near path derives once per (line, warp).
struct NearLine {
  double nu0, A1, g2, a2, inv_alpha, inv_a2, y, Acore, xc2;
};

// Wing value amp*V(d) for one point with the regime chosen per thread (divergent; near path and test hook only).
// Valid for r^2 >= xc2-region complement, i.e. the caller handles the core separately.
__device__ __forceinline__ double wing_value(double d, const NearLine &L)
{
  const double q = d * d;
  const double r2 = (L.a2 > 0.0) ? (q + L.g2) * L.inv_a2 : __longlong_as_double(0x7ff0000000000000LL);
  if (r2 >= kR1) {
    return gh1_acc(0.0, d, L.A1, L.g2);
  } else if (r2 >= kR2) {
    return gh2_acc(0.0, d, L.A1, L.g2 - 0.5 * L.a2, 2.0 * L.a2 * L.g2, L.A1 * L.a2);
  } else if (r2 >= kR3) {
    const double c3 = L.A1 * (1.0 / 3.0);
    return gh3_acc(0.0, d, L.g2, L.g2 - 1.5 * L.a2, 6.0 * L.a2 * L.g2, 2.0 * c3, c3, L.A1 * L.a2);
  } else {
    return L.A1 * gh6_shape(q, L.g2, L.a2);
  }
}

// core switch in x^2 for a line of damping y: series where x^2 < xc2.  Beyond the ring r^2 = 44 the 6-point rule is
// good to 3.7e-8 except that no wing rule carries the Gaussian term exp(-x^2); for y < 1e-8 that term is still
// > 1e-10 of K at r^2 = 44, so the series region is widened to x^2 < -ln(1e-10 y) (capped by the 32-term table).
__device__ __forceinline__ double core_xc2(double y)
{
  double xc2 = kRc - y * y;
  if (y < 1e-8) xc2 = fmax(xc2, -log(1e-10 * fmax(y, 1e-300)));
  xc2 = fmin(xc2, kXcapSq);
  return xc2 > 0.0 ? xc2 : 0.0;
}

}  // namespace hk
