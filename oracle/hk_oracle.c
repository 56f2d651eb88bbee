/* oracle/hk_oracle.c — CPU ORACLE.  TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * A plain, slow, double-precision restatement of what the HELIOS-K hot path computes
 * (Grimm & Heng 2015, arXiv:1503.03806; citations are PAPER.md line numbers):
 *
 *   kappa(nu_j) = sum_i (S_i/m) * Phi_i(nu_j)          eq. 16, summed over lines
 *   Phi = sqrt(ln2/pi) H_V / Gamma_D,  H_V = Re w(u+ia) eq. 19
 *   per-bin k-distribution: sort, y_k uniform, resample  eqs. 14-15
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may
 * call this.  It shares no code, header, table or constant generator with the CUDA path under
 * paper_1503_03806_b200/, and neither imports the other.
 *
 * The paper's method evaluates H_V approximately (Algorithm 916 / Gauss-Hermite);
 * the quantity being approximated has a plain definition, so the oracle is that definition: H_V is
 * evaluated here by an independent routine accurate to ~1e-13 (no regime approximations):
 *   - Laplace continued fraction of w(z) for |z|^2 >= 64 or y >= 0.5,
 *   - Taylor expansion in y about the real axis, w(x) = exp(-x^2) + 2i/sqrt(pi) Dawson(x), otherwise.
 * Neither formula appears in the CUDA path.
 *
 * Pins (tests/test_oracle_*.py, all run without a GPU): mpmath 50-digit evaluation of
 * exp(-z^2) erfc(-iz) on a lattice (tests/golden/faddeeva_golden.csv) and brute-force mpmath.quad of
 * the Voigt convolution integral; K(0,y)=erfcx(y); K(x,y->0)=exp(-x^2); symmetry; Lorentz asymptote;
 * Gaussian and Lorentzian limits of V; unit area; numpy + scipy.special.wofz brute force of a whole
 * small opacity function with the window computed independently; numpy sort + interp for the
 * k-distribution; numpy leggauss for the nodes.  No function here is "parity unpinned".
 *
 * Readings of the paper taken here are listed in DESIGN.md ("Readings"): G1-G4, A3-A9.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define ORC_OK 0
#define ORC_ERR_INVALID (-1)
#define ORC_ERR_NOMEM (-3)

/* physical constants, CGS */
#define ORC_C_LIGHT 2.99792458e10      /* cm/s */
#define ORC_K_B 1.380649e-16           /* erg/K */
#define ORC_AMU 1.66053906660e-24      /* g */
#define ORC_C2 1.4388                  /* cm K, hc/k_B as BASELINE.json config 4 writes it */
#define ORC_T0 296.0                   /* K */

static const long double SQRTPI_L = 1.7724538509055160272981674833411451828L;
static const long double PI_L = 3.1415926535897932384626433832795028842L;

/* ------------------------------------------------------------------------------------------
 * Gauss-Legendre nodes and weights on (0,1): roots of P_n by Newton, mapped g = (1+t)/2.
 * (north_star: "cumulative resampling at Gauss-Legendre g-points".)  Ascending in g.
 * ---------------------------------------------------------------------------------------- */
static void legendre_l(int n, long double t, long double *p, long double *dp)
{
    long double p0 = 1.0L, p1 = t;
    if (n == 0) { *p = 1.0L; *dp = 0.0L; return; }
    for (int k = 2; k <= n; k++) {
        long double pk = ((2 * k - 1) * t * p1 - (k - 1) * p0) / k;
        p0 = p1; p1 = pk;
    }
    *p = p1;
    *dp = n * (t * p1 - p0) / (t * t - 1.0L);
}

static int gauss_legendre_l(int n, long double *g, long double *w)
{
    if (n < 1) return ORC_ERR_INVALID;
    for (int i = 0; i < n; i++) {
        /* Chebyshev-like first guess for the i-th root counted from the top, then Newton */
        long double t = cosl(PI_L * (i + 0.75L) / (n + 0.5L)), p, dp;
        for (int it = 0; it < 100; it++) {
            legendre_l(n, t, &p, &dp);
            long double dt = p / dp;
            t -= dt;
            if (fabsl(dt) < 1e-19L) break;
        }
        legendre_l(n, t, &p, &dp);
        int k = n - 1 - i;                       /* ascending order */
        g[k] = 0.5L * (1.0L + t);
        w[k] = 1.0L / ((1.0L - t * t) * dp * dp); /* = (2/((1-t^2)P'^2)) / 2 for the (0,1) map */
    }
    return ORC_OK;
}

int orc_gauss_legendre(int n, double *g, double *w)
{
    if (n < 1 || n > 4096 || !g || !w) return ORC_ERR_INVALID;
    long double *gl = (long double *)malloc(sizeof(long double) * 2 * (size_t)n);
    if (!gl) return ORC_ERR_NOMEM;
    int rc = gauss_legendre_l(n, gl, gl + n);
    for (int i = 0; i < n; i++) { g[i] = (double)gl[i]; w[i] = (double)gl[n + i]; }
    free(gl);
    return rc;
}

/* ------------------------------------------------------------------------------------------
 * Dawson's integral F(x) = exp(-x^2) * int_0^x exp(t^2) dt = int_0^x exp(t^2 - x^2) dt, x >= 0,
 * by composite 24-point Gauss-Legendre on panels of width <= 0.5 (integrand positive: no cancellation).
 * ---------------------------------------------------------------------------------------- */
#define DAW_NG 24
static long double daw_g[DAW_NG], daw_w[DAW_NG];
static int daw_ready = 0;
__attribute__((constructor)) static void daw_init(void)
{
    gauss_legendre_l(DAW_NG, daw_g, daw_w);
    daw_ready = 1;
}

static long double dawson_l(long double x)
{
    if (x == 0.0L) return 0.0L;
    int np = (int)ceill(x / 0.5L);
    if (np < 1) np = 1;
    long double h = x / np, sum = 0.0L, x2 = x * x;
    for (int p = 0; p < np; p++) {
        long double a = p * h, s = 0.0L;
        for (int q = 0; q < DAW_NG; q++) {
            long double t = a + h * daw_g[q];
            s += daw_w[q] * expl(t * t - x2);
        }
        sum += s * h;
    }
    return sum;
}

/* ------------------------------------------------------------------------------------------
 * K(x,y) = Re w(x+iy),  w(z) = exp(-z^2) erfc(-iz)   (H_V of eq. 19 with u=x, a=y)
 * ---------------------------------------------------------------------------------------- */

/* Laplace continued fraction  w(z) = (i/sqrt(pi)) / (z - (1/2)/(z - 1/(z - (3/2)/(z - ...)))),
 * evaluated backward from depth n with tail f = z.  With f = fr + i fi:
 *   (k/2)/f = (k/2)(fr - i fi)/|f|^2, so  z - (k/2)/f = (x - t fr) + i (y + t fi),  t = (k/2)/|f|^2.
 * Every nested imaginary part stays >= y > 0 (no cancellation in Re w).
 * Finally w = (i/sqrt(pi)) (fr - i fi)/|f|^2  =>  Re w = fi / (sqrt(pi) |f|^2). */
static double K_cf(double x, double y, int depth)
{
    long double fr = x, fi = y;
    for (int k = depth; k >= 1; k--) {
        long double den = fr * fr + fi * fi;
        long double t = (0.5L * k) / den;
        fr = (long double)x - t * fr;
        fi = (long double)y + t * fi;
    }
    long double den = fr * fr + fi * fi;
    return (double)(fi / (SQRTPI_L * den));
}

/* Taylor expansion about the real axis:  w(x+iy) = sum_n w^(n)(x) (iy)^n / n!,
 *   w(x)  = exp(-x^2) + (2i/sqrt(pi)) F(x),   F = Dawson
 *   w'(x) = -2x w + 2i/sqrt(pi),   w^(n+1) = -2x w^(n) - 2n w^(n-1). */
static double K_taylor(double x, double y)
{
    long double xl = x, yl = y;
    long double w0r = expl(-xl * xl), w0i = 2.0L / SQRTPI_L * dawson_l(xl);
    long double w1r = -2.0L * xl * w0r, w1i = -2.0L * xl * w0i + 2.0L / SQRTPI_L;
    /* c = (iy)^n/n! ; start n=1: c = i y */
    long double cr = 0.0L, ci = yl;
    long double sum = w0r + (w1r * cr - w1i * ci);
    long double wmr = w0r, wmi = w0i, wnr = w1r, wni = w1i;
    for (int n = 1; n < 400; n++) {
        long double wxr = -2.0L * xl * wnr - 2.0L * n * wmr;
        long double wxi = -2.0L * xl * wni - 2.0L * n * wmi;
        /* c *= (i y)/(n+1) */
        long double tr = -ci * yl / (n + 1), ti = cr * yl / (n + 1);
        cr = tr; ci = ti;
        long double add = wxr * cr - wxi * ci;
        sum += add;
        wmr = wnr; wmi = wni; wnr = wxr; wni = wxi;
        long double mag = (fabsl(wxr) + fabsl(wxi)) * (fabsl(cr) + fabsl(ci));
        if (n > 8 && mag < 1e-24L * fabsl(sum)) break;
    }
    return (double)sum;
}

double orc_faddeeva_re(double x, double y)
{
    x = fabs(x);                      /* K(-x,y) = K(x,y) */
    double r2 = x * x + y * y;
    if (!(y > 0.0)) {                 /* y = 0: on the real axis Re w = exp(-x^2) */
        return exp(-x * x);
    }
    if (r2 >= 64.0 || y >= 0.5) {
        int depth;
        if (r2 >= 1.0e4) depth = 8;
        else if (r2 >= 1.0e3) depth = 10;
        else if (r2 >= 200.0) depth = 14;
        else if (r2 >= 64.0) depth = 24;
        else {                         /* |z|^2 < 64, y >= 0.5: slow convergence ~ 1/y^2 */
            depth = (int)ceil(260.0 / (y * y));
            if (depth < 60) depth = 60;
        }
        return K_cf(x, y, depth);
    }
    return K_taylor(x, y);
}

void orc_voigt_K(const double *x, const double *y, int64_t n, double *out)
{
#pragma omp parallel for schedule(dynamic, 256)
    for (int64_t i = 0; i < n; i++) out[i] = orc_faddeeva_re(x[i], y[i]);
}

/* ------------------------------------------------------------------------------------------
 * Line parameters (BASELINE.json configs; DESIGN.md readings)
 *   alpha = (nu0/c) sqrt(2 kB T / m)      [ = Gamma_D / sqrt(ln 2) ]
 *   gamma = gamma0 * P_atm * (296/T)^n    [ eq. 20, pressure term only ]
 *   S(T)  = S                                              if E_low == NULL
 *         = S q_ratio exp(-c2 E (1/T - 1/296)) (1-exp(-c2 nu0/T)) / (1-exp(-c2 nu0/296))    eq. 18
 * Window: j_lo = max(0, ceil(((nu0-cutoff)-nu_min)/dnu)), j_hi = min(N-1, floor(((nu0+cutoff)-nu_min)/dnu)).
 * ---------------------------------------------------------------------------------------- */
typedef struct {
    double nu0, amp, alpha, gamma;
    int64_t jlo, jhi;
    int64_t src;
} orc_line;

static int cmp_line(const void *a, const void *b)
{
    const orc_line *p = (const orc_line *)a, *q = (const orc_line *)b;
    if (p->nu0 < q->nu0) return -1;
    if (p->nu0 > q->nu0) return 1;
    return (p->src > q->src) - (p->src < q->src);
}

double orc_line_strength(double S, double nu0, double E_low, double T, double q_ratio)
{
    double boltz = exp(-ORC_C2 * E_low * (1.0 / T - 1.0 / ORC_T0));
    double stim;
    if (nu0 == 0.0) stim = ORC_T0 / T;              /* limit of the ratio as nu0 -> 0 */
    else stim = (-expm1(-ORC_C2 * nu0 / T)) / (-expm1(-ORC_C2 * nu0 / ORC_T0));
    return S * q_ratio * boltz * stim;
}

void orc_window(double nu0, double nu_min, int64_t N, double dnu, double cutoff, int64_t *jlo, int64_t *jhi)
{
    double a = ceil(((nu0 - cutoff) - nu_min) / dnu);
    double b = floor(((nu0 + cutoff) - nu_min) / dnu);
    if (a < 0.0) a = 0.0;
    if (b > (double)(N - 1)) b = (double)(N - 1);
    if (a > 9.0e18) a = 9.0e18;
    if (b < -9.0e18) b = -9.0e18;
    *jlo = (int64_t)a;
    *jhi = (int64_t)b;
}

int64_t orc_count_evals(const double *nu0, int64_t n, double nu_min, int64_t N, double dnu, double cutoff)
{
    int64_t tot = 0;
    for (int64_t i = 0; i < n; i++) {
        int64_t lo, hi;
        orc_window(nu0[i], nu_min, N, dnu, cutoff, &lo, &hi);
        if (hi >= lo) tot += hi - lo + 1;
    }
    return tot;
}

/* Voigt profile value V(dnu; alpha, gamma) = K(dnu/alpha, gamma/alpha)/(alpha sqrt(pi)).
 * alpha == 0 (nu0 == 0) or x, y beyond 1e150: the Lorentzian gamma/(pi (dnu^2+gamma^2)) (A9). */
double orc_voigt_V(double dv, double alpha, double gamma)
{
    if (alpha > 0.0) {
        double x = dv / alpha, y = gamma / alpha;
        if (fabs(x) < 1e150 && y < 1e150)
            return orc_faddeeva_re(x, y) / (alpha * 1.7724538509055160273);
    }
    return gamma / (3.14159265358979323846 * (dv * dv + gamma * gamma));
}

/* kappa_out[k] = kappa(nu_{js[k]}) for an arbitrary list of grid indices.  Lines may come in any order. */
int orc_opacity_points_rel(const double *nu0_in, const double *S, const double *gamma0, const double *gamma_self,
                           const double *A21, const double *delta, const double *n_T, const double *E_low,
                           int64_t n_lines, double T, double P_atm, double self_fraction, double abundance, double nu_min,
                           int64_t N, double dnu, double cutoff, double cutoff_widths, double mass_amu, double q_ratio,
                           const int64_t *js, int64_t n_js, double *kappa_out);

/* Full line physics: eq. 20 with the natural width A21/(4 pi c), air and self
 * broadening, P_self = self_fraction * P ("in equal proportions (P_self = 0.5 P)"), P0 = 1 atm:
 *     gamma = A21/(4 pi c) + (T/T0)^(-n) [ gamma_air (P - P_self)/P0 + gamma_self P_self/P0 ]
 * and eq. 21: nu0 -> nu0 + delta P/P0, the shifted centre replacing nu0 everywhere after it (profile
 * centre, Doppler width, window, eq. 18: DESIGN.md reading C2).  NULL gamma_self: no self term (P_self = 0); NULL A21:
 * no natural width; NULL delta: no shift.  abundance X multiplies the species' opacity (kappa = sum_s X_s kappa_s,
 * PAPER.md:133-135). */
int orc_opacity_points_full(const double *nu0_in, const double *S, const double *gamma0, const double *gamma_self,
                            const double *A21, const double *delta, const double *n_T, const double *E_low,
                            int64_t n_lines, double T, double P_atm, double self_fraction, double abundance, double nu_min,
                            int64_t N, double dnu, double cutoff, double mass_amu, double q_ratio, const int64_t *js,
                            int64_t n_js, double *kappa_out)
{
    return orc_opacity_points_rel(nu0_in, S, gamma0, gamma_self, A21, delta, n_T, E_low, n_lines, T, P_atm, self_fraction,
                                  abundance, nu_min, N, dnu, cutoff, 0.0, mass_amu, q_ratio, js, n_js, kappa_out);
}

/* The same with a RELATIVE line-wing cutoff ("an ad hoc cutoff of 500 Lorentz widths"):
 * cutoff_widths > 0 truncates line i at min(cutoff, cutoff_widths * gamma_i), gamma_i the Lorentz half-width of eq. 20
 * (reading C5: the absolute cutoff stays as an upper bound; pass a large one for a purely relative cutoff).
 * cutoff_widths == 0: the absolute cutoff alone. */
int orc_opacity_points_rel(const double *nu0_in, const double *S, const double *gamma0, const double *gamma_self,
                           const double *A21, const double *delta, const double *n_T, const double *E_low,
                           int64_t n_lines, double T, double P_atm, double self_fraction, double abundance, double nu_min,
                           int64_t N, double dnu, double cutoff, double cutoff_widths, double mass_amu, double q_ratio,
                           const int64_t *js, int64_t n_js, double *kappa_out)
{
    if (n_lines < 0 || !(T > 0.0) || !(P_atm > 0.0) || !(dnu > 0.0) || !(cutoff > 0.0) || N <= 0 || !(mass_amu > 0.0) ||
        n_js < 0 || (n_js > 0 && (!js || !kappa_out)))
        return ORC_ERR_INVALID;
    if (n_lines > 0 && (!nu0_in || !S || !gamma0)) return ORC_ERR_INVALID;
    for (int64_t k = 0; k < n_js; k++)
        if (js[k] < 0 || js[k] >= N) return ORC_ERR_INVALID;
    double m_g = mass_amu * ORC_AMU;
    double vth = sqrt(2.0 * ORC_K_B * T / m_g) / ORC_C_LIGHT;     /* alpha = nu0 * vth */
    orc_line *L = (orc_line *)malloc(sizeof(orc_line) * (size_t)(n_lines > 0 ? n_lines : 1));
    if (!L) return ORC_ERR_NOMEM;
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n_lines; i++) {
        double nT = n_T ? n_T[i] : 0.5;
        double nu0 = delta ? nu0_in[i] + delta[i] * P_atm : nu0_in[i];                    /* eq. 21, P0 = 1 atm */
        double P_self = gamma_self ? self_fraction * P_atm : 0.0;
        double press = gamma0[i] * (P_atm - P_self) + (gamma_self ? gamma_self[i] * P_self : 0.0);
        L[i].nu0 = nu0;
        L[i].alpha = nu0 * vth;
        L[i].gamma = pow(ORC_T0 / T, nT) * press;                                          /* eq. 20, pressure terms */
        if (A21) L[i].gamma += A21[i] / (4.0 * 3.14159265358979323846 * ORC_C_LIGHT);     /* natural width */
        double s = E_low ? orc_line_strength(S[i], nu0, E_low[i], T, q_ratio) : S[i];
        L[i].amp = abundance * s / m_g;
        double cut = cutoff;
        if (cutoff_widths > 0.0 && cutoff_widths * L[i].gamma < cut) cut = cutoff_widths * L[i].gamma;
        orc_window(nu0, nu_min, N, dnu, cut, &L[i].jlo, &L[i].jhi);
        L[i].src = i;
    }
    int sorted = 1;
    for (int64_t i = 1; i < n_lines; i++)
        if (L[i - 1].nu0 > L[i].nu0) { sorted = 0; break; }
    if (!sorted) qsort(L, (size_t)n_lines, sizeof(orc_line), cmp_line);
    double slack = cutoff + 4.0 * dnu;
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t k = 0; k < n_js; k++) {
        int64_t j = js[k];
        double nu = nu_min + (double)j * dnu;
        /* candidates: first line with nu0 >= nu - slack; the exact test is the index window below */
        int64_t lo = 0, hi = n_lines;
        while (lo < hi) {
            int64_t mid = lo + (hi - lo) / 2;
            if (L[mid].nu0 < nu - slack) lo = mid + 1; else hi = mid;
        }
        long double acc = 0.0L;
        for (int64_t i = lo; i < n_lines && L[i].nu0 <= nu + slack; i++) {
            if (j < L[i].jlo || j > L[i].jhi) continue;
            acc += (long double)L[i].amp * (long double)orc_voigt_V(nu - L[i].nu0, L[i].alpha, L[i].gamma);
        }
        kappa_out[k] = (double)acc;
    }
    free(L);
    return ORC_OK;
}

int orc_opacity_points(const double *nu0, const double *S, const double *gamma0, const double *n_T, const double *E_low,
                       int64_t n_lines, double T, double P_atm, double nu_min, int64_t N, double dnu, double cutoff,
                       double mass_amu, double q_ratio, const int64_t *js, int64_t n_js, double *kappa_out)
{
    return orc_opacity_points_full(nu0, S, gamma0, NULL, NULL, NULL, n_T, E_low, n_lines, T, P_atm, 0.0, 1.0, nu_min, N, dnu,
                                   cutoff, mass_amu, q_ratio, js, n_js, kappa_out);
}

/* kappa_out[j - j_begin] for j in [j_begin, j_end). */
int orc_opacity(const double *nu0, const double *S, const double *gamma0, const double *n_T, const double *E_low,
                int64_t n_lines, double T, double P_atm, double nu_min, int64_t N, double dnu, double cutoff,
                double mass_amu, double q_ratio, int64_t j_begin, int64_t j_end, double *kappa_out)
{
    if (j_begin < 0 || j_end > N || j_end < j_begin || !kappa_out) return ORC_ERR_INVALID;
    int64_t n = j_end - j_begin;
    int64_t *js = (int64_t *)malloc(sizeof(int64_t) * (size_t)(n > 0 ? n : 1));
    if (!js) return ORC_ERR_NOMEM;
    for (int64_t k = 0; k < n; k++) js[k] = j_begin + k;
    int rc = orc_opacity_points(nu0, S, gamma0, n_T, E_low, n_lines, T, P_atm, nu_min, N, dnu, cutoff, mass_amu, q_ratio,
                                js, n, kappa_out);
    free(js);
    return rc;
}

/* ------------------------------------------------------------------------------------------
 * k-distribution per bin (eqs. 14-15): ascending sort; the k-th sorted value sits
 * at y_k = (k + 1/2)/ppb (equal delta-y = 1/N_nu); linear interpolation at the Gauss-Legendre nodes,
 * clamped to the end values (A7).  k_out is [n_bins][n_g], row-major.
 * ---------------------------------------------------------------------------------------- */
static int cmp_double(const void *a, const void *b)
{
    double p = *(const double *)a, q = *(const double *)b;
    return (p > q) - (p < q);
}

int orc_kdist(const double *kappa, int64_t n_points, int64_t ppb, int n_g, double *k_out)
{
    if (!kappa || !k_out || n_points <= 0 || ppb <= 0 || n_g < 1 || n_points % ppb != 0) return ORC_ERR_INVALID;
    int64_t n_bins = n_points / ppb;
    double *g = (double *)malloc(sizeof(double) * 2 * (size_t)n_g);
    if (!g) return ORC_ERR_NOMEM;
    int rc = orc_gauss_legendre(n_g, g, g + n_g);
    if (rc != ORC_OK) { free(g); return rc; }
    int fail = 0;
#pragma omp parallel for schedule(dynamic, 4)
    for (int64_t b = 0; b < n_bins; b++) {
        double *s = (double *)malloc(sizeof(double) * (size_t)ppb);
        if (!s) { fail = 1; continue; }
        memcpy(s, kappa + b * ppb, sizeof(double) * (size_t)ppb);
        qsort(s, (size_t)ppb, sizeof(double), cmp_double);
        for (int q = 0; q < n_g; q++) {
            double p = g[q] * (double)ppb - 0.5, v;
            if (p <= 0.0) v = s[0];
            else if (p >= (double)(ppb - 1)) v = s[ppb - 1];
            else {
                int64_t k = (int64_t)floor(p);
                double f = p - (double)k;
                v = s[k] + f * (s[k + 1] - s[k]);
            }
            k_out[b * n_g + q] = v;
        }
        free(s);
    }
    free(g);
    return fail ? ORC_ERR_NOMEM : ORC_OK;
}
