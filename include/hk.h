/* hk.h — C ABI of the B200-native HELIOS-K hot path (Grimm & Heng 2015, arXiv:1503.03806).
 *
 * The library computes, entirely in its own sm_100a CUDA kernels,
 *
 *   (1) the line-by-line opacity function on a uniform wavenumber grid
 *         kappa(nu_j) = sum_i (S_i(T)/m) * Phi_i(nu_j),      nu_j = nu_min + j*dnu,  j = 0..N-1
 *       eq. 16 with the Voigt profile Phi = sqrt(ln2/pi) H_V / Gamma_D of eq. 19
 *       (PAPER.md:176-183), H_V = Re w(u+ia) evaluated by an Algorithm-916-type series near the line
 *       core and n-point Gauss-Hermite quadrature in the wings, every line truncated
 *       at an absolute line-wing cutoff, lines looped serially and grid points in
 *       parallel with kappa accumulated in registers;
 *   (2) the k-distribution of kappa in fixed-width bins: per-bin ascending sort, equal delta-y = 1/N_nu
 *       (eqs. 14-15), resampled at n_g Gauss-Legendre nodes on (0,1)
 *       (BASELINE.json north_star); the paper's own Chebyshev fit is hk_kdist_cheb, and the
 *       transmission function of eq. 5 is hk_transmission / hk_transmission_direct.
 *
 * Conventions
 *   - Every pointer marked "device" is a CUDA device pointer (e.g. torch .data_ptr()); "host" is host memory.
 *     All arrays are contiguous float64 unless stated.  Inputs are read-only and caller-owned; outputs are
 *     caller-allocated and are OVERWRITTEN — with one exception, kappa_out under hk_params.accumulate = 1 (a mixture's
 *     running sum), which is added to.
 *   - Calls enqueue work on `stream` (a cudaStream_t passed as void*; NULL = the legacy default stream) and
 *     return without synchronising, except where stated; the caller synchronises before reading results.
 *     Scratch memory is taken from the library's own stream-ordered CUDA memory pool (one per device, kept for reuse)
 *     and returned to it on the same stream (hk_opacity_noalloc excepted: it allocates nothing, see there).
 *   - Return value: HK_OK (0) or a negative HK_ERR_* code; hk_strerror() names it; after HK_ERR_CUDA,
 *     hk_last_cuda_error() returns the CUDA runtime's message.  No exceptions.
 *   - State the library keeps.  Per host thread: the last-error string, the hk_set_timing() switch with its events, and
 *     the copy stream of hk_opacity_host.  Per device, created on first use under a lock and kept for the life of the
 *     process: the memory pool (hk_trim() returns its idle memory to the driver), the kernels' shared-memory attributes
 *     and launch grids, and the Chebyshev projection matrices of hk_kdist_cheb.  Calls may come from several host threads
 *     and, after cudaSetDevice, for several devices; an hk_ctx belongs to the device and stream it was created on and must
 *     not be used from two threads at once.
 *   - Units: wavenumbers in cm^-1, T in K, P in atm (1 atm = 1.01325 bar), mass in amu,
 *     S in cm/molecule, kappa in cm^2/g.
 *   - There is no CPU fallback: without a CUDA device every compute entry point returns HK_ERR_CUDA.
 */
#ifndef HK_H_
#define HK_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define HK_OK 0
#define HK_ERR_INVALID (-1)     /* bad argument (see each function) */
#define HK_ERR_CUDA (-2)        /* CUDA runtime error; see hk_last_cuda_error() */
#define HK_ERR_NOMEM (-3)       /* device or host allocation failed */
#define HK_ERR_UNSORTED (-4)    /* hk_lines_check_sorted(): nu0 is not ascending */
#define HK_ERR_UNSUPPORTED (-5) /* valid request outside the implemented range (e.g. points per bin > 16384) */

#define HK_FP64 0
#define HK_FP32 1               /* optional FP32 variant (north_star; bar 1e-4): see hk_opacity */

/* Line list, structure of arrays, all DEVICE pointers, n_lines entries each.
 * These are the fields of a HITRAN/HITEMP record that the simplified broadening law of
 * BASELINE.json uses (PAPER.md:164-191 lists the full record). */
typedef struct {
  const double *nu0;    /* line centre nu_0, cm^-1                                                  */
  const double *S;      /* line strength, cm/molecule: at T if E_low == NULL, else at T0 = 296 K     */
  const double *gamma0; /* Lorentz HWHM at 296 K and 1 atm, cm^-1/atm                                */
  const double *n_T;    /* temperature exponent n_coll of eq. 20, or NULL for 0.5 on every line      */
  const double *E_low;  /* lower-state energy, cm^-1, or NULL: no S(T) scaling (eq. 18 not applied)  */
  /* full line physics of eqs. 20-21; each may be NULL (term absent): */
  const double *gamma_self; /* self-broadening HWHM alpha_self at 296 K, 1 atm, cm^-1/atm (gamma0 is then alpha_air) */
  const double *A21;        /* Einstein A coefficient, s^-1: natural width A21/(4 pi c)                      */
  const double *delta;      /* pressure-induced shift delta_shift, cm^-1/atm (eq. 21)                        */
} hk_lines;

typedef struct {
  double mass_amu;      /* molecular mass m (one species per call), amu; > 0                          */
  double q_ratio;       /* Q(296 K)/Q(T) of eq. 18; used only when E_low != NULL                      */
  int precision;        /* HK_FP64 (bar 1e-6) or HK_FP32 (bar 1e-4): arithmetic of the far-wing rules, see hk_opacity */
  int lines_sorted;     /* 1: caller guarantees nu0 ascending, as HITRAN/HITEMP files are (not re-checked; see
                           hk_lines_check_sorted()).  0: the library checks on the device (synchronises the
                           stream) and, if needed, works on a copy ordered by nu0; inputs are never modified */
  void *stream;         /* cudaStream_t, or NULL                                                      */
  double self_fraction; /* P_self/P of eq. 20 (the paper takes 0.5), in [0,1]; used only when
                           gamma_self != NULL                                                         */
  double abundance;     /* X_s: the species' opacity is multiplied by it (kappa = sum_s X_s kappa_s);
                           0 means 1, so that a zero-initialised tail keeps the one-species behaviour          */
  double cutoff_widths; /* relative line-wing cutoff ("500 Lorentz widths"): > 0 truncates line i at
                           min(cutoff, cutoff_widths * gamma_i), gamma_i the Lorentz half-width of eq. 20 at (T, P);
                           0: the absolute cutoff alone.  The absolute `cutoff` stays the upper bound (and sizes the line
                           ranges the kernels scan: keep it near cutoff_widths * max gamma for speed)            */
  int accumulate;       /* 0: kappa_out is overwritten.  1: X_s kappa_s is ADDED to kappa_out — the species are summed
                           BEFORE the sort, as PAPER.md:135 requires; the first species of a mixture passes 0     */
} hk_params;

/* N = llround((nu_max - nu_min)/dnu): number of grid points nu_j = nu_min + j*dnu, j < N. Host only. */
int64_t hk_grid_size(double nu_min, double nu_max, double dnu);

/* Opacity function (steps a1-a4 of DESIGN.md: line prep, tile plan, Voigt accumulation, kappa store).
 *
 *   gamma_i = gamma0_i * P_atm * (296/T)^n_i                      eq. 20, pressure term
 *   alpha_i = (nu0_i/c) sqrt(2 k_B T/m)  [= Gamma_D/sqrt(ln 2)]
 *   S_i(T)  = S_i, or eq. 18 (T0 = 296 K in the last denominator) when E_low != NULL, with
 *             c2 = hc/k_B = 1.4388 cm K
 *   window  : line i contributes to j_lo(i) <= j <= j_hi(i)  (cutoff -> min(cutoff, cutoff_widths*gamma_i) when
 *             prm->cutoff_widths > 0),
 *             j_lo = max(0, ceil(((nu0-cutoff)-nu_min)/dnu)), j_hi = min(N-1, floor(((nu0+cutoff)-nu_min)/dnu))
 *             (inclusive, decided in index space; hard truncation, no renormalisation)
 *   kappa_j = sum_{i in window} (S_i(T)/(m*amu)) * K(x_ij, y_i)/(alpha_i sqrt(pi)),  x = (nu_j-nu0)/alpha, y = gamma/alpha
 *
 * K = Re w(x+iy) is evaluated to <= 2.5e-7 relative error: Algorithm-916-type series for x^2+y^2 < 44,
 * 6/3/2-point Gauss-Hermite rules beyond 44 / 280 / 3200, and from max(3600, 4100 y) the 1-point rule with the
 * shifted denominator x^2 + y^2 - 3/2.  Degenerate lines: nu0 <= 0 (alpha = 0) is a pure
 * Lorentzian; gamma = 0 (gamma0 = 0 and no natural width) is the pure Doppler profile exp(-x^2)/(alpha sqrt(pi)).
 *
 * Full line physics, active per optional array of hk_lines:
 *   gamma_i = A21_i/(4 pi c) + (296/T)^n_i [ gamma0_i (P - P_self) + gamma_self_i P_self ],  P_self = self_fraction * P   eq. 20
 *   nu0_i  -> nu0_i + delta_i * P_atm                                                                                    eq. 21
 * (P0 = 1 atm).  The shifted centre replaces nu0 everywhere downstream (profile centre, Doppler width, window, eq. 18).
 * The list is NOT re-ordered for the shift: a1 shifts every centre itself and builds its line-range tables from the unshifted,
 * ordered centres with a halo of max_i |delta_i| * P_atm; the one-shot call finds that maximum by a small reduction
 * (synchronises the stream once), a context finds it once at hk_create.  lines_sorted refers to the unshifted nu0.
 * Mixtures: call once per species with prm->abundance = X_s and prm->accumulate = 1 from the second species on; the
 * k-distribution of the sum is then taken by hk_kdist (adding k-distributions instead would be the correlated-k
 * approximation).
 *
 * prm->precision = HK_FP32 (north_star's optional FP32 variant, max relative error <= 1e-4): the same ladder with the
 * switches at 44 / 64 / 300 / max(400, 400 y) (each rule <= 4e-5 from exact K); the 1-, 2- and 3-point rules — every 32-point
 * group outside the line's 3-point radius, ~99.7 % of all evaluations — run in FP32 (distances from an integer + fraction
 * split of the line centre in grid units, a float partial sum per 32 lines added to FP64 accumulators); the 6-point
 * rule and the series near the centre stay FP64 (and so do the three grid points on either side of every line centre,
 * where the float distance would cancel), as do line prep, the index windows and kappa_out.  A line whose amplitude
 * S gamma/(pi m) is more than 2^-127 below the largest of the lines of its batch of 32 that reach the same 256-point span
 * flushes to zero in this mode.  The float wing rules keep their denominators inside the float range by construction: on
 * grids finer than 1.3e-5 cm^-1 the FP64 band around every centre widens to 4e-5 cm^-1, and a line whose window reaches
 * beyond 5e4 cm^-1 from its centre takes the 3-point rule throughout; a cutoff beyond 2e6 cm^-1 is refused in this mode
 * (HK_ERR_UNSUPPORTED; any cutoff wider than the grid and the list already means "no cutoff").
 *
 * kappa_out: device, N doubles, overwritten.  Lines outside [nu_min, nu_max) still contribute if within the
 * cutoff.  n_lines == 0 gives kappa == 0.
 * HK_ERR_INVALID: NULL lines/prm/kappa_out or (n_lines > 0 and NULL nu0/S/gamma0); n_lines < 0; T, P_atm, dnu,
 * cutoff, mass_amu not > 0 or not finite; N < 1 or N > 2^30; precision unknown; abundance or cutoff_widths < 0 or
 * not finite;
 * self_fraction outside [0,1] when gamma_self != NULL.
 * Asynchronous on prm->stream (synchronises once when lines_sorted = 0).  nu0 must be ascending when
 * lines_sorted = 1 (see hk_lines_check_sorted). */
int hk_opacity(const hk_lines *lines, int64_t n_lines, double T, double P_atm, double nu_min, double nu_max,
               double dnu, double cutoff, double *kappa_out, const hk_params *prm);

/* End-to-end form with HOST buffers (what bench.py's `e2e` times): copies the line arrays host -> device, runs
 * hk_opacity and, when k_host_out != NULL, hk_kdist(bin_width, n_g), copies kappa (when kappa_host_out != NULL) and the
 * k-table device -> host, and waits for the stream.  The Voigt accumulation runs as six (far kernel, near kernel) launch pairs
 * over ranges of the grid, each on a library-owned stream of its own, and every range of kappa is copied back on a further
 * stream as soon as it is final, while the later ranges are still being computed.  Every array of lines_host is a HOST pointer (pinned memory makes
 * the copies asynchronous to the host but is not required); kappa_host_out: host [N] or NULL; k_host_out: host
 * [n_bins*n_g] or NULL (then bin_width and n_g are ignored); at least one output is required.  Device memory comes from
 * the library's pool.  With prm->accumulate = 1 kappa_host_out is also an INPUT (the running sum of the mixture, copied
 * host -> device first) and must not be NULL.  Errors as hk_opacity / hk_kdist.  Synchronous. */
int hk_opacity_host(const hk_lines *lines_host, int64_t n_lines, double T, double P_atm, double nu_min, double nu_max,
                    double dnu, double cutoff, double *kappa_host_out, double bin_width, int n_g, double *k_host_out,
                    const hk_params *prm);

/* hk_opacity for callers that must not allocate device memory.
 *
 * Who this is for.  Some programs cannot let a library take memory from the CUDA driver at the moment they call it: a
 * serving or training process that handed all of the GPU's memory to its own arena at start-up (a cudaMalloc, or the
 * growth of this library's pool, would then fail or eat into what the arena was promised); a latency-bound loop that
 * shares the device with other running streams (an allocation may take driver locks or make the device wait); a
 * deployment whose memory is audited after start-up and where later allocation calls are forbidden outright.
 * hk_opacity() takes its work space — the packed per-line records of step a1 and the line-range tables of step a2 — from
 * the library's memory pool, which grows through the driver on demand; this entry point runs the same kernels with that
 * work space in a fixed array compiled into the library (`static __device__`, 256-byte aligned) instead.
 *
 * The price and the limits.  The array is HK_NOALLOC_SCRATCH_BYTES (about 11.2 MiB) and exists on every GPU on which
 * the process has loaded this library, used or not, until the process exits.  It holds at most HK_NOALLOC_MAX_LINES
 * lines and a grid of at most HK_NOALLOC_MAX_POINTS points; a larger request returns HK_ERR_UNSUPPORTED and
 * hk_last_cuda_error() says which limit was passed and by how much.  (A longer list can be fed in ordered pieces of
 * at most HK_NOALLOC_MAX_LINES lines with prm->accumulate = 1 from the second piece on; a longer grid in ranges.)
 * Two services of hk_opacity() need an allocation and a host wait and are therefore refused here, also with
 * HK_ERR_UNSUPPORTED: prm->lines_sorted must be 1 (no order check, no ordered copy: pass nu0 ascending), and
 * lines->delta must be NULL (no pressure shift, eq. 21).  hk_set_timing() has no effect on this call.
 *
 * Arguments, results, units, the remaining error codes and both precisions are those of hk_opacity(); for the same
 * inputs the output is bit-for-bit the same.  The caller still supplies every input and kappa_out as device memory
 * of its own.  The call enqueues on prm->stream and returns without waiting.  It makes no cudaMalloc / cudaFree /
 * pool call and calls no library routine that allocates device memory.
 *
 * First call on each device.  The first call a process makes on a given device (with that device current) looks up
 * the device address of the array, sets the kernels' shared-memory attributes and sizes their grids, and lets the
 * CUDA runtime load the kernels; later calls on that device only launch.  Make that first call during start-up, before
 * any stream capture is begun.
 *
 * One array, shared.  Every call on a device — from any host thread, on any stream — uses the same array, and the array
 * keeps what the previous call left in it.  Nothing in it is trusted from call to call: every record and table entry a
 * call reads is written by that call first, and the tile-ticket counters that must start at zero are cleared by the
 * call's first kernel.  Because the array is shared, two of these calls must not overlap on the GPU: issue them on one
 * stream, or order them with events.  Calls that overlap race on the array and give wrong results without any error.
 * hk_opacity() and the other entry points do not touch the array and may run beside it. */
#define HK_NOALLOC_MAX_LINES 65536
#define HK_NOALLOC_MAX_POINTS 4194304
#define HK_NOALLOC_SCRATCH_BYTES (HK_NOALLOC_MAX_LINES * 176 + 196864)
int hk_opacity_noalloc(const hk_lines *lines, int64_t n_lines, double T, double P_atm, double nu_min, double nu_max,
                       double dnu, double cutoff, double *kappa_out, const hk_params *prm);

/* Synchronous check that a device nu0 array is ascending (what lines_sorted = 1 promises).
 * Returns HK_OK, HK_ERR_UNSORTED, or an error.  Blocks until the stream is idle. */
int hk_lines_check_sorted(const double *nu0_device, int64_t n_lines, void *stream);

/* Metric denominator: sum_i (j_hi(i) - j_lo(i) + 1) over lines with a non-empty window.  HOST array. */
int64_t hk_count_evals(const double *nu0_host, int64_t n_lines, double nu_min, int64_t N, double dnu, double cutoff);

/* k-distribution (steps a5-a6): bins of ppb = llround(bin_width/dnu) consecutive points, aligned at index 0.
 *   s = ascending sort of kappa[b*ppb : (b+1)*ppb];  y_k = (k + 1/2)/ppb   (eq. 15: delta-y = 1/N_nu)
 *   k_out[b][q] = linear interpolation of (y_k, s_k) at the q-th Gauss-Legendre node g_q on (0,1),
 *                 clamped to s_0 / s_{ppb-1} outside [y_0, y_{ppb-1}].
 * kappa: device [n_points], values >= 0 (or +inf), no NaN.  k_out: device [n_bins*n_g], row-major by bin, overwritten.
 * HK_ERR_INVALID: NULL pointers, n_points < 1, dnu or bin_width not > 0, bin_width/dnu not an integer within 1e-9,
 * n_points not a multiple of ppb, n_g < 1 or > 128.   HK_ERR_UNSUPPORTED: ppb > 16384.   Asynchronous. */
int hk_kdist(const double *kappa, int64_t n_points, double dnu, double bin_width, int n_g, double *k_out, void *stream);

/* the paper's own resampling: per bin, least-squares fit of ln kappa(y) with n_c
 * Chebyshev polynomials of t = 2y - 1 at the cell centres y_k = (k + 1/2)/ppb of the sorted bin,
 *   minimise sum_k ( sum_n C_n T_n(2 y_k - 1) - ln max(s_k, 1e-300) )^2 ,
 * "solving A C = D" by Q-R decomposition.  The design matrix A is the same for every bin, so it is factored once per
 * (ppb, n_c) (Householder Q-R in long double on the host; P = R^-1 Q^T kept on the device for the life of the process;
 * that first call synchronises); each call is the sort kernel, which also stores ln of the sorted values in a scratch
 * array from the library's pool, and one projection kernel C = D P^T.  The paper is
 * silent on kappa = 0: ln is taken of max(kappa, 1e-300).
 * coef_out: device [n_bins*n_c], row-major by bin, overwritten.  k_out: device [n_bins*n_g] or NULL — when given, the
 * Gauss-Legendre k-table of hk_kdist is written by the same launch (n_g is ignored when k_out is NULL).
 * HK_ERR_INVALID: as hk_kdist, or NULL coef_out, n_c < 1, n_c > 64, n_c > ppb.  HK_ERR_UNSUPPORTED: ppb > 16384. */
int hk_kdist_cheb(const double *kappa, int64_t n_points, double dnu, double bin_width, int n_c, double *coef_out, int n_g,
                  double *k_out, void *stream);

/* The projection matrix hk_kdist_cheb uses, P[n][k] (row-major, n_c x ppb) with C = P D: host arithmetic only (no GPU
 * needed), for inspection and tests.  P_host_out: HOST [n_c*ppb].  HK_ERR_INVALID: NULL, n_c < 1 or > 64, ppb < n_c or
 * > 16384. */
int hk_cheb_projection(int ppb, int n_c, double *P_host_out);

/* kappa_y_out[b][i] = exp( sum_n coef[b][n] T_n(2 y_i - 1) ): the resampled k-distribution function of every bin at the
 * abscissae y (device [n_y], in [0,1]), by the Clenshaw recurrence.  coef: device [n_bins*n_c]; kappa_y_out: device
 * [n_bins*n_y], overwritten.  HK_ERR_INVALID: NULL, n_bins < 1, n_c < 1 or > 64, n_y < 1.  Asynchronous. */
int hk_cheb_eval(const double *coef, int64_t n_bins, int n_c, const double *y, int n_y, double *kappa_y_out, void *stream);

/* transmission function of every bin for n_m column masses m~ [g cm^-2] (eq. 5, PAPER.md:74-80;
 * "computing T for 1000 values of m~"):
 *   hk_transmission         T[b][m] = int_0^1 exp(-kappa(y) m~) dy = sum_q w_q exp(-k_table[b][q] m~_m)   (Lebesgue side)
 *                           with the n_g-point Gauss-Legendre weights whose nodes hk_kdist sampled;
 *   hk_transmission_direct  T[b][m] = (1/Delta x) int exp(-kappa(x) m~) dx = mean over the bin's ppb grid points of
 *                           exp(-kappa_j m~_m)                                                              (Riemann side).
 * k_table: device [n_bins*n_g]; kappa: device [n_points], finite; mcol: device [n_m], >= 0; T_out: device [n_bins*n_m],
 * row-major by bin, overwritten.  HK_ERR_INVALID: NULL, n_bins < 1, n_g < 1 or > 128, n_m < 1, or the bin arguments as
 * in hk_kdist.  Asynchronous. */
int hk_transmission(const double *k_table, int64_t n_bins, int n_g, const double *mcol, int n_m, double *T_out, void *stream);
int hk_transmission_direct(const double *kappa, int64_t n_points, double dnu, double bin_width, const double *mcol, int n_m,
                           double *T_out, void *stream);

/* n_g Gauss-Legendre nodes g (ascending) and weights w on (0,1), sum w = 1.  HOST arrays of n_g doubles.
 * HK_ERR_INVALID for n_g < 1, n_g > 4096 or NULL. */
int hk_gauss_legendre(int n_g, double *g, double *w);

/* Test hook: out[i] = K(x[i], y[i]) = Re w(x+iy) through the device Voigt routine of hk_opacity (same regime
 * switches; precision = HK_FP32: the FP32 variant's switches and float 1-/2-point rules).  x, y, out: device [n];
 * y > 0.  HK_ERR_INVALID: NULL, n < 0, unknown precision.  Asynchronous. */
int hk_voigt_K(const double *x, const double *y, int64_t n, double *out, int precision, void *stream);

/* Persistent-context form for T-P sweeps ("repeat this calculation for multiple combinations of
 * temperature and pressure"): the line list is bound once, scratch is kept between calls.
 * hk_create copies nothing when nu0 is ascending: the hk_lines device arrays must outlive the context; with
 * lines_sorted = 0 and an unordered list the context owns an ordered copy (made once).  A pressure-shift field (delta !=
 * NULL) costs nothing extra per call (see hk_opacity); hk_create synchronises the stream once to find max |delta|.
 * self_fraction, abundance, cutoff_widths and accumulate are taken from prm at hk_create. */
typedef struct hk_ctx hk_ctx;
int hk_create(const hk_lines *lines, int64_t n_lines, const hk_params *prm, hk_ctx **out);
int hk_opacity_ctx(hk_ctx *ctx, double T, double P_atm, double q_ratio, double nu_min, double nu_max, double dnu,
                   double cutoff, double *kappa_out);
int hk_destroy(hk_ctx *ctx);

/* Measurement helper: runs a dependent-FMA FP64 loop on every SM and returns the achieved FP64
 * thread-instructions per second (the "alu" roofline denominator of bench.py, measured live).  Synchronous. */
int hk_fp64_peak(double *inst_per_s_out, void *stream);

/* Likewise for the FP32 pipe (dependent FFMA; the roofline denominator of the FP32 variant).  Synchronous. */
int hk_fp32_peak(double *inst_per_s_out, void *stream);

/* Measurement helper (roofline numerator of bench.py): how many line-point evaluations of the workload fall in each
 * regime of the device Voigt routine (switches of `precision`), decided per POINT on r^2 = x^2 + y^2 as hk_voigt_K does:
 * counts_out[0..4] = 1-point, 2-point, 3-point, 6-point Gauss-Hermite, series.  Their sum equals hk_count_evals().
 * gamma = gamma0 * P_atm * (296/T)^0.5 (n_T = 0.5), alpha = (nu0/c) sqrt(2 k_B T/m).  HOST arrays, host arithmetic,
 * O(n_lines).  HK_ERR_INVALID on NULL, non-positive T, P_atm, mass_amu, dnu, cutoff, N, or unknown precision. */
int hk_regime_census(const double *nu0_host, const double *gamma0_host, int64_t n_lines, double T, double P_atm,
                     double mass_amu, double nu_min, int64_t N, double dnu, double cutoff, int precision,
                     int64_t counts_out[5]);

/* Per-stage device time of the last hk_opacity / hk_opacity_ctx call on this thread, in milliseconds, measured
 * with CUDA events on the call's stream: [0] line prep (a1, with the lookup tables of a2), [1] Voigt accumulation, far
 * kernel (1-, 2- and 3-point rule, writes kappa), [2] Voigt accumulation, near kernel (6-point rule and series, adds to
 * kappa); a3 + a4 = [1] + [2].  Enabled by hk_set_timing(1) (off by default; the switch is per host thread).  The timed call stays asynchronous: it only
 * records the events; hk_last_stage_ms() waits for the last one (synchronous) and must be called before the next timed
 * call. */
int hk_set_timing(int on);
int hk_last_stage_ms(float ms_out[3]);

/* Returns the idle memory of the current device's pool to the driver (scratch of a config-4-sized call is otherwise kept
 * for reuse for the life of the process).  Synchronises the device. */
int hk_trim(void);

const char *hk_strerror(int code);
const char *hk_last_cuda_error(void);
const char *hk_version(void);

#ifdef __cplusplus
}
#endif
#endif /* HK_H_ */
