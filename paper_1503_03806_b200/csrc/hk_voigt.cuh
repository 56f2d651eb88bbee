// hk_voigt.cuh — device Voigt-profile arithmetic for sm_100a (FP64 pipe; no tensor cores: not a contraction).
//
// The profile value of one line at one grid point (eq. 19),
//     V(d) = K(d/alpha, gamma/alpha) / (alpha sqrt(pi)),     K(x,y) = H_V = Re w(x+iy)
// is evaluated in one of five regimes chosen on r^2 = x^2 + y^2 (PAPER.md:197 gives the three-regime
// structure and calls its switch points "trial-and-error"; DESIGN.md §4 derives these):
//
//   r^2 >= max(3600, 4100 y) : 1-point rule with shifted denominator          5 FP64 + 1 MUFU per point
//   r^2 >= 3200  : 2-point Gauss-Hermite                                       7 FP64 + 1 MUFU
//   r^2 >= 280   : 3-point Gauss-Hermite ("third-order", Letchworth & Benner) 11 FP64 + 1 MUFU
//   r^2 >= 44    : 6-point Gauss-Hermite                                      22 FP64 + 3 MUFU
//   else         : Algorithm-916-type series (Zaghloul & Ali 2012), step a = 0.7, 16 terms   83 FP64 + 1 MUFU
// (the kernels switch between the last two at x^2 = 44.15 - y^2, inside the band where both are valid: kSeriesPad)
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

// 1-point rule with the shifted denominator, K = (y/sqrt(pi)) / (x^2 + y^2 - 3/2)  (V = A1/(d^2 + gamma^2 - 1.5 alpha^2)):
// the second term of w(z) ~ (i/sqrt(pi)) (1/z)(1 + 1/(2 z^2) + 3/(4 z^4) + ...) folded into the Lorentzian's denominator.  Its
// relative error is 1.5/x^4 + 2 y^2/r^4 (checked against the oracle: tests/test_rule_accuracy.py), so it serves from
// r^2 >= max(kR1a, kR1b y) at the cost of the plain 1-point rule (which needs r^2 >= 6e6 for the same accuracy).
constexpr double kR1a = 3600.0, kR1b = 4100.0;  // 1.2e-7 + 1.2e-7 <= 2.4e-7
constexpr double kR2 = 3200.0;  // 2-point rule             (2.4e-7)
constexpr double kR3 = 280.0;   // 3-point rule             (2.4e-7)
constexpr double kRc = 44.0;    // 6-point rule from here (3.7e-8); series below
// FP32 variant (hk_params.precision = HK_FP32; north_star: "optional FP32 path", bar 1e-4): the same ladder with the
// switches moved in to where each rule is <= 4e-5 from exact K (1-point 1.5/x^2, 2-point
// 2.8e-5 at 300, 3-point 2.2e-5 at 64); the 1- and 2-point rules (the far kernel: ~99 % of all evaluations) run in FP32.
constexpr double kR1fa = 400.0, kR1fb = 400.0;  // shifted 1-point rule from r^2 >= max(400, 400 y)   (9.4e-6 + 1.3e-5)
constexpr double kR2f = 300.0;  // 2-point rule             (2.8e-5)
constexpr double kR3f = 64.0;   // 3-point rule             (2.2e-5)
constexpr double kXgCapSq = 270.0;  // the Gaussian term is never added beyond the 6-point region (exp(-270) = 5e-118)
constexpr double kTinyY = 1.0e-8;   // below this damping the wing rules miss a visible exp(-x^2) beyond r^2 = 44

constexpr double kPi = 3.14159265358979323846;
constexpr double kInvPi = 0.31830988618379067153776753;
constexpr double kSqrtPi = 1.772453850905516027298167;
constexpr double kInvSqrtPi = 0.5641895835477562869480795;

// Algorithm-916-type series constants, step a = 0.7 (truncation error 1.1e-8 relative, uniform in y)
constexpr double kA = 0.7;
constexpr int kTerms = 16;                                // a n <= x + 4.4 for x <= sqrt(44)
constexpr double k2AoverPi = 0.4456338406573069401528745; // 2a/pi
constexpr double kAoverPi = 0.2228169203286534700764373;  // a/pi

// 6-point Gauss-Hermite: t_k^2 and normalised weights w_k/sqrt(pi) of the three +- pairs
constexpr double kT6sq0 = 0.1901635091934881328718554, kW6_0 = 0.4088284695560292260885378;
constexpr double kT6sq1 = 1.784492748543251591186722, kW6_1 = 0.08861574604191452748085588;
constexpr double kT6sq2 = 5.525343742263260275941422, kW6_2 = 0.002555784402056246430606291;

// r^2 from which the (shifted) 1-point rule serves a line of damping y
__device__ __host__ __forceinline__ double r1_sq(double y, bool f32)
{
  const double a = f32 ? kR1fa : kR1a, b = (f32 ? kR1fb : kR1b) * y;
  return a > b ? a : b;
}

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
// 1/x to ~2^-80 (two Newton steps): for the few per-line reciprocals that feed the series
__device__ __forceinline__ double rcp_nr2(double x)
{
  double r = rcp_nr(x);
  double e = fma(-x, r, 1.0);
  return fma(r, e, r);
}

// ---- wing rules: contribution amp * V(d) added to acc --------------------------------------------------
// 1-point: A1/(d^2+g2s), A1 = amp*gamma/pi, g2s = gamma^2 - 1.5 alpha^2 (shifted denominator, see kR1a)
__device__ __forceinline__ double gh1_acc(double acc, double d, double A1, double g2)
{
  double D = fma(d, d, g2);
  return fma(A1, rcp_nr(D), acc);
}
// the same for TWO points with one reciprocal, 1/(D0 D1): 10 FP64 + 1 MUFU per pair — the FP64 count of two gh1_acc, half
// the MUFU.RCP64H (the XU unit, 16 lanes/SM, is the far kernel's second-busiest pipe)
__device__ __forceinline__ void gh1_acc2(double &a0, double &a1, double d0, double d1, double A1, double g2)
{
  const double D0 = fma(d0, d0, g2), D1 = fma(d1, d1, g2);
  const double t = A1 * rcp_nr(D0 * D1);
  a0 = fma(t, D1, a0);
  a1 = fma(t, D0, a1);
}
// the same for FOUR points with one reciprocal, 1/(D0 D1 D2 D3), through the cross products c02 = D0 D2, c13 = D1 D3:
// A1/D0 = (t c13) D2, A1/D1 = (t c02) D3, A1/D2 = (t c13) D0, A1/D3 = (t c02) D1 with t = A1/(c02 c13).  20 FP64 + 1 MUFU
// per four points: the FP64 count of two pairs, a quarter of the MUFU.RCP64H of four single evaluations.
__device__ __forceinline__ void gh1_acc4(double &a0, double &a1, double &a2, double &a3, double d0, double d1, double d2,
                                         double d3, double A1, double g2)
{
  const double D0 = fma(d0, d0, g2), D1 = fma(d1, d1, g2), D2 = fma(d2, d2, g2), D3 = fma(d3, d3, g2);
  const double c02 = D0 * D2, c13 = D1 * D3;
  const double t = A1 * rcp_nr(c02 * c13);
  const double u0 = t * c13, u1 = t * c02;
  a0 = fma(u0, D2, a0);
  a1 = fma(u1, D3, a1);
  a2 = fma(u0, D0, a2);
  a3 = fma(u1, D1, a3);
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
// ---- FP32 wing rules (far kernel of the FP32 variant): TWO points per reciprocal, 1/(D0 D1) by one MUFU.RCP (1 ulp),
// so that the MUFU unit (16 lanes/SM) does not bound the FP32 pipe (128 lanes/SM).  d^4 products stay far inside the
// float range: the 2-point rule is only used for |d| < 200 alpha.
__device__ __forceinline__ float rcpf(float x)
{
  float r;
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
  return r;
}
__device__ __forceinline__ void gh1_acc2f(float &a0, float &a1, float d0, float d1, float A1, float g2)
{
  const float D0 = fmaf(d0, d0, g2), D1 = fmaf(d1, d1, g2);
  const float t = A1 * rcpf(D0 * D1);
  a0 = fmaf(t, D1, a0);
  a1 = fmaf(t, D0, a1);
}
__device__ __forceinline__ void gh2_acc2f(float &a0, float &a1, float d0, float d1, float A1, float e2, float f2, float A1a2)
{
  const float E0 = fmaf(d0, d0, e2), E1 = fmaf(d1, d1, e2);
  const float D0 = fmaf(E0, E0, f2), D1 = fmaf(E1, E1, f2);
  const float B0 = fmaf(A1, E0, A1a2), B1 = fmaf(A1, E1, A1a2);
  const float r = rcpf(D0 * D1);
  a0 = fmaf(B0 * D1, r, a0);
  a1 = fmaf(B1 * D0, r, a1);
}
// ---- packed FP32 pairs (sm_100: fma / mul / add .f32x2 -> SASS FFMA2 / FMUL2 / FADD2, two floats per 64-bit register and
// per issue slot).  The FP32 far kernel is issue-bound, and its points already come in pairs. ----
typedef unsigned long long f32x2;
__device__ __forceinline__ f32x2 pk2(float lo, float hi)
{
  f32x2 r;
  asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
  return r;
}
__device__ __forceinline__ void upk2(f32x2 v, float &lo, float &hi) { asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v)); }
__device__ __forceinline__ f32x2 fma2(f32x2 a, f32x2 b, f32x2 c)
{
  f32x2 r;
  asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c));
  return r;
}
__device__ __forceinline__ f32x2 mul2(f32x2 a, f32x2 b)
{
  f32x2 r;
  asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
  return r;
}
__device__ __forceinline__ f32x2 add2(f32x2 a, f32x2 b)
{
  f32x2 r;
  asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
  return r;
}
// 1-point rule on FOUR points (two packed pairs p, q) with one reciprocal, 1/(D0 D1 D2 D3): with the cross products
// c = (D0 D2, D1 D3) and u = A1 r (c.hi, c.lo), the four terms A1/D_k are u * (D2, D3) and u * (D0, D1): no operand swaps.
// 10 issue slots + 1 MUFU.RCP for four evaluations (the scalar pair form: 9 + 1 for two).  D^4 stays inside the float range:
// D <= cutoff^2 ~ 1e4, and D >= (3 dnu)^2 (the FP64 guard band of a1 keeps the far kernel three grid steps off every centre).
__device__ __forceinline__ void gh1_acc4f(f32x2 &ap, f32x2 &aq, f32x2 dp, f32x2 dq, float A1, f32x2 g2g2)
{
  const f32x2 Dp = fma2(dp, dp, g2g2), Dq = fma2(dq, dq, g2g2);
  const f32x2 c = mul2(Dp, Dq);
  float c0, c1;
  upk2(c, c0, c1);
  const float t = A1 * rcpf(c0 * c1);
  const f32x2 u = mul2(pk2(t, t), pk2(c1, c0));
  ap = fma2(u, Dq, ap);
  aq = fma2(u, Dp, aq);
}
// 2-point rule on a packed pair with one reciprocal: 7 issue slots + 1 MUFU.RCP (scalar form: 13 + 1)
__device__ __forceinline__ void gh2_acc2p(f32x2 &a, f32x2 d, f32x2 A1A1, f32x2 e2e2, f32x2 f2f2, f32x2 wa2)
{
  const f32x2 E = fma2(d, d, e2e2);
  const f32x2 D = fma2(E, E, f2f2);
  const f32x2 B = fma2(A1A1, E, wa2);
  float D0, D1;
  upk2(D, D0, D1);
  const float r = rcpf(D0 * D1);
  a = fma2(mul2(B, pk2(D1, D0)), pk2(r, r), a);
}
// 3-point rule in float (FP32 variant: from r^2 >= 64), one reciprocal per point (R D ~ d^6 would leave the float range in
// a product over two points)
__device__ __forceinline__ float gh3_accf(float acc, float d, float g2, float e3, float f3, float c0, float c3, float c3a)
{
  const float R = fmaf(d, d, g2), E = fmaf(d, d, e3);
  const float D = fmaf(E, E, f3), B = fmaf(c3, E, c3a);
  const float num = fmaf(c0, D, B * R);
  return fmaf(num, rcpf(R * D), acc);
}
// per-line constants of one +-t pair of the 6-point rule: E = q + e, value = (cE * E + c0) / (E^2 + f)
struct GhPair {
  double e, f, cE, c0;
};
__device__ __forceinline__ GhPair gh_pair_consts(double A1, double g2, double a2, double tsq, double wn)
{
  GhPair p;
  p.e = g2 - tsq * a2;
  p.f = 4.0 * tsq * a2 * g2;
  p.cE = 2.0 * wn * A1;
  p.c0 = p.cE * (2.0 * tsq * a2);
  return p;
}
__device__ __forceinline__ double gh_pair_val(double q, const GhPair &p)
{
  double E = q + p.e;
  double D = fma(E, E, p.f);
  return fma(p.cE, E, p.c0) * rcp_nr(D);
}
struct Gh6 {
  GhPair p0, p1, p2;
};
__device__ __forceinline__ Gh6 gh6_consts(double A1, double g2, double a2)
{
  Gh6 g;
  g.p0 = gh_pair_consts(A1, g2, a2, kT6sq0, kW6_0);
  g.p1 = gh_pair_consts(A1, g2, a2, kT6sq1, kW6_1);
  g.p2 = gh_pair_consts(A1, g2, a2, kT6sq2, kW6_2);
  return g;
}
// 6-point: amp * V(d), 3 x (DADD + 4 DFMA/DMUL + Newton reciprocal) + 2 DADD = 22 FP64 + 3 MUFU
__device__ __forceinline__ double gh6_val(double q, const Gh6 &g)
{
  return gh_pair_val(q, g.p0) + gh_pair_val(q, g.p1) + gh_pair_val(q, g.p2);
}

// exp(x) for -700 < x < 700 (no overflow / underflow / NaN handling: the series calls it on [-300, 10]).  n = rint(x log2 e)
// by the magic-number add, r = x - n ln2 in two pieces, a degree-11 Taylor polynomial on |r| <= ln2/2 (remainder 6e-15)
// whose coefficients are operands from the constant bank, 2^n added to the exponent field: 16 FP64 + 3 integer
// instructions.  The library exp() spends about as many FP64 instructions but twice as many issue slots (its 64-bit
// immediates arrive by UMOV pairs, and it guards the range): the near kernel is issue-bound, not FP64-bound.
__constant__ double kExpTaylor[12] = {1.0, 1.0, 0.5, 1.0 / 6, 1.0 / 24, 1.0 / 120, 1.0 / 720, 1.0 / 5040, 1.0 / 40320,
                                      1.0 / 362880, 1.0 / 3628800, 1.0 / 39916800};
template <int DEG>
__device__ __forceinline__ double exp_poly(double x)
{
  const double kMagic = 6755399441055744.0;  // 1.5 * 2^52
  const double t = fma(x, 1.4426950408889634074, kMagic);
  const int n = __double2loint(t);
  const double nd = t - kMagic;
  double r = fma(nd, -6.93147180369123816490e-01, x);  // ln2 high part (its low 21 bits are zero)
  r = fma(nd, -1.90821492927058770002e-10, r);         // ln2 low part
  double p = kExpTaylor[DEG];
#pragma unroll
  for (int k = DEG - 1; k >= 0; --k) p = fma(p, r, kExpTaylor[k]);
  return __hiloint2double(__double2hiint(p) + (n << 20), __double2loint(p));
}
__device__ __forceinline__ double exp_fast(double x) { return exp_poly<11>(x); }
// the series' own exponentials: degree 8 (remainder (ln2/2)^9/9! = 2e-10 relative; the series itself is truncated at 1.1e-8)
__device__ __forceinline__ double exp_series(double x) { return exp_poly<8>(x); }

// sin(t)^2 for 0 <= t < 1e4 (the series calls it with t = x y <= 44): k = rint(t/pi) by the magic-number add, r = t - k pi in
// two pieces (|r| <= pi/2; the sign of sin(t) = (-1)^k sin(r) does not matter for the square), sin(r) = r P(r^2) with the
// Taylor coefficients to degree 19 (remainder 3e-16) from the constant bank.  Relative accuracy holds for small t (the term
// sin^2(xy)/y -> x^2 y as y -> 0 needs it).  14 FP64 instructions; the library sinpi costs about twice the issue slots.
__constant__ double kSinTaylor[10] = {1.0, -1.0 / 6, 1.0 / 120, -1.0 / 5040, 1.0 / 362880, -1.0 / 39916800, 1.0 / 6227020800.0,
                                      -1.0 / 1307674368000.0, 1.0 / 355687428096000.0, -1.0 / 121645100408832000.0};
template <int STEPS>
__device__ __forceinline__ double sin_sq_poly(double t)
{
  const double kMagic = 6755399441055744.0;  // 1.5 * 2^52
  const double kd = fma(t, 0.31830988618379067154, kMagic) - kMagic;
  double r = fma(kd, -3.14159265160560607910e+00, t);  // pi high part (low 26 bits zero: kd * it is exact for kd < 2^26)
  r = fma(kd, -1.98418714791870343106e-09, r);         // pi middle part
  r = fma(kd, -1.14423774522196636802e-17, r);         // pi low part
  const double q = r * r;
  double p = kSinTaylor[STEPS];
#pragma unroll
  for (int k = STEPS - 1; k >= 0; --k) p = fma(p, q, kSinTaylor[k]);
  return q * p * p;
}
__device__ __forceinline__ double sin_sq_fast(double t) { return sin_sq_poly<9>(t); }
// the series' own: sin(r)/r to degree 12 in r (remainder (pi/2)^14/15! = 4e-10 relative)
__device__ __forceinline__ double sin_sq_series(double t) { return sin_sq_poly<6>(t); }

// ---- core: Algorithm-916-type series (restated in DESIGN.md §4) ---------------------------
//   K(x,y) = exp(-x^2) [ erfcx(y) cos(2xy) + (2a/pi) sin^2(xy)/y - (2a/pi) y cos(2xy) S1(y)
//                        + (a/pi) y sum_{n=1..16} W_n (p^n + p^-n) ],
//   W_n = exp(-a^2 n^2)/(a^2 n^2 + y^2),  S1 = sum_n W_n,  p = exp(2 a x)
// (exp(-(an-x)^2) + exp(-(an+x)^2) = exp(-x^2) exp(-a^2 n^2) (p^n + p^-n)).  With cos(2xy) = 1 - 2 sin^2(xy) the bracket is
//   E0 + sin^2(xy) B2 + (a/pi) y sum,     E0 = erfcx(y) - (2a/pi) y S1,   B2 = (2a/pi)/y - 2 E0.
// y is a per-line constant: E0, B2 and the 16 weights W_n are computed once per line (SeriesLine + a 16-entry table in
// shared memory, read by broadcast in the series loop, one LDS.128 per two terms) and carry the line's amplitude.
// C_n = p^n + p^-n advances by the three-term recurrence C_{n+2} = ((p + 1/p)^2 - 2) C_n - C_{n-2} (forward-stable: the
// growing solution dominates) in two independent chains (odd and even n), so a term is 2 DFMA.
// p^16 <= exp(1.4 * 6.7 * 16) = 1e65: no overflow for x <= 6.7.
__constant__ double kSeriesEn[kTerms] = {  // exp(-a^2 n^2), n = 1..16
    0.612626394184416069,    0.140858420921044996,    0.0121551783299149372,   0.000393669040655078211,
    4.78511739212900909e-6,  2.18295779512547921e-8,  3.73757132794426203e-11, 2.40173478162095945e-14,
    5.79231288539485792e-18, 5.24288566336346394e-22, 1.78106663475709136e-26, 2.27081292202639651e-31,
    1.08661064074598053e-36, 1.95145238029537775e-42, 1.31532589485746453e-48, 3.32736305418299429e-55};

struct SeriesLine {
  double inv_alpha;  // x = |d| / alpha
  double y;          // gamma/alpha (>= 1e-200: line prep floors it)
  double Aay;        // A (a/pi) y,    A = amp/(alpha sqrt(pi)): the result is amp * V(d)
  double AE0;        // A E0
  double AB2;        // A B2
};

// Per-line constants of the series, by ONE thread: writes W_1..W_16 to W[0..15] and returns the rest.
__device__ __forceinline__ SeriesLine series_line_setup(double y, double inv_y, double erfcx_y, double Acore, double inv_alpha,
                                                        double *W)
{
  const double y2 = y * y;
  double S1 = 0.0;
#pragma unroll
  for (int n = 1; n <= kTerms; ++n) {
    const double w = kSeriesEn[n - 1] * rcp_nr2(fma(kA * kA * (double)n, (double)n, y2));
    W[n - 1] = w;
    S1 += w;
  }
  const double E0 = fma(-k2AoverPi * y, S1, erfcx_y);
  SeriesLine L;
  L.inv_alpha = inv_alpha;
  L.y = y;
  L.Aay = Acore * (kAoverPi * y);
  L.AE0 = Acore * E0;
  L.AB2 = Acore * fma(k2AoverPi, inv_y, -2.0 * E0);
  return L;
}

// amp * V(d) by the series, valid for |d| / alpha <= 6.7.  Every term is even in x (exp(-x^2), cosh(2 a n x), sin^2(x y)), so the
// signed x = d / alpha serves, and x is not clamped: callers discard the lanes beyond the series region (there the result
// is meaningless, possibly inf or NaN, and never stored) — fabs + fmin cost five issue slots per evaluation in an
// issue-bound kernel (profiles/r03_near_instruction_mix.txt).  About 83 FP64 instructions: two exponentials (13 each),
// reciprocal (3), recurrence and sums (35), sin^2 (13), the rest head and tail.
__device__ __forceinline__ double series_val(double d, const SeriesLine &L, const double *W)
{
  const double x = d * L.inv_alpha;
  const double ex2 = exp_series(-x * x);
  const double p = exp_series((2.0 * kA) * x);
  const double s2 = sin_sq_series(x * L.y);
  const double s2c = p + rcp_nr(p);  // 2 cosh(2 a x) = C_1
  const double t2 = fma(s2c, s2c, -2.0);
  double Com = s2c, Co = s2c, Cem = 2.0, Ce = t2, so = 0.0, se = 0.0;  // C_{-1} = C_1, C_0 = 2, C_2 = C_1^2 - 2
#pragma unroll
  for (int i = 0; i < kTerms / 2; ++i) {
    const double2 w = *reinterpret_cast<const double2 *>(W + 2 * i);
    so = fma(w.x, Co, so);
    se = fma(w.y, Ce, se);
    const double Con = fma(t2, Co, -Com), Cen = fma(t2, Ce, -Cem);
    Com = Co; Co = Con;
    Cem = Ce; Ce = Cen;
  }
  const double head = fma(s2, L.AB2, L.AE0);
  return ex2 * fma(L.Aay, so + se, head);
}

// Where the kernels switch between the series and the 6-point rule: the series is valid for every x <= 6.7 and the 6-point
// rule wherever x^2 + y^2 >= 44, so any switch with 44 - y^2 <= x^2 <= 44.89 is valid; a1 puts it at x^2 = 44.15 - y^2, in
// index space (the band is wide enough that no rounding of the FP64 index arithmetic can leave it).
constexpr double kSeriesPad = 0.15;
// series region of a line of damping y: x^2 < xc2 = 44 - y^2 (none for y >= sqrt(44))
__device__ __host__ __forceinline__ double core_xc2(double y)
{
  const double xc2 = kRc - y * y;
  return xc2 > 0.0 ? xc2 : 0.0;
}
// No wing rule carries the Gaussian term exp(-x^2).  For y < 1e-8 it is still > 1e-10 of K beyond the series region, so
// the 6-point rule adds it out to x^2 = xg2 = -ln(1e-10 y)  (K = exp(-x^2) + wing + O(y^2)); 0 = never.
__device__ __host__ __forceinline__ double gauss_xg2(double y)
{
  if (!(y < kTinyY)) return 0.0;
  const double v = -log(1e-10 * (y > 1e-300 ? y : 1e-300));
  return v < kXgCapSq ? v : kXgCapSq;
}

}  // namespace hk
