/*
 * ll_oracle.c — CPU ORACLE for the batched LISA MBHB log-likelihood.  TEST INFRASTRUCTURE ONLY.
 *
 * Plain, slow, obviously-correct restatement of what the hot path computes, written from
 * /root/reference/PAPER.md (arXiv:2111.01064) and the readings listed in DESIGN.md §3.
 * It shares NO code, header, table or constant with the CUDA library under
 * paper_2111_01064_b200/csrc/ and includes nothing from include/.  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may call it.
 *
 * Arithmetic: inputs and outputs are fp64; intermediates and every accumulator are `long double`
 * (x87 80-bit), sums are plain sequential loops in the order the paper writes them, trig is
 * glibc sinl/cosl on the phase in radians.  No blocking, fusion, skipping or reordering beyond
 * the band mask, which is part of the definition (reading R10).
 *
 * What follows the paper:
 *   log L = -1/2 <d-h|d-h> = -1/2(<d|d> + <h|h> - 2<d|h>)                     Eq. 2
 *   <a|b> = 4 Re sum_{ch} int a~* b~ / S_n df                                  Eq. 3
 *   h~_lm = A_lm(f) exp(-i phi_lm(f))                                          Eq. 7
 *   h~^{A,E}(f) = sum_lm T^{A,E}_lm h~_lm(f)                                   Eq. 9
 *   r = h/h0 = r0 + r1 (f - f_b)                                               Eq. 11
 *   Z[d,h] = 4 Re sum_b A0 r0* + A1 r1*                                        Eq. 14-16
 *   Z[h,h] = 4 sum_b B0 |r0|^2 + 2 B1 Re[r0 r1*]                               Eq. 17-19
 *   r0, r1 = intercept and slope of the complex line across the bin edges
 * What does not (PAPER.md is silent; BASELINE.json north_star/configs + DESIGN.md readings):
 *   natural cubic spline of amplitude and phase on sparse nodes (R1, R2), the TaylorF2 stand-in
 *   waveform and its taper (R9), the band mask (R10), the weights W_k = 4 df w_k / S_n (R4).
 *
 * Pins (tests/test_oracle_pins.py, all -m "not gpu"): SciPy natural CubicSpline, dense Gaussian
 * elimination, linear/cubic reproduction; closed-form <h|h> under a flat PSD (+ Euler-Maclaurin term)
 * and mpmath sums; log L = 0 at d = h; 1/D, phi_c scalings; brute-force numpy/mpmath sums on tiny
 * inputs; summary-data partition exactness; het exactness for r linear in f and its known B2
 * deficit; het == full at h = h0; the frequency-dependent-T path against the constant-T path, a template
 * whose T is linear in f against direct numpy evaluation, SciPy on tiny inputs; t_lm against SciPy's spline
 * derivative and the stand-in's analytic d Psi/df; three channels with per-channel weights against SciPy + numpy channel
 * by channel, the closed-form <h|h> under three different flat PSDs, additivity over channels and equality with the
 * shared-weight path when the rows are equal; the linear phase term outside the spline (t_shift) against splining the
 * full phase (a natural spline reproduces linear functions) and SciPy.  No function here is "parity unpinned".
 *
 * Layouts (all row-major, fp64):
 *   d, h, h0_dense, noise : [n_c][n_f][2]  (re, im)
 *   W                     : [n_f] (w_rows = 1: one PSD for every channel) or [n_c][n_f] (w_rows = n_c: W^c_k =
 *                           4 df w_k / S^c_n(f_k), each TDI channel with its own noise PSD; Eq. 3 sums over A, E, T and
 *                           "A=E identical, T different")
 *   amp, phase            : [n_w][n_m][n_nodes]   (phase in radians)
 *   tf                    : [n_w][n_m][n_c][2]
 *   tf_nodes              : [n_w][n_m][n_c][n_nodes][2]   (frequency-dependent transfer function, Eq. 8-9)
 *   band                  : [n_w][2] (f_lo, f_hi) or NULL
 *   t_shift               : [n_w] seconds or NULL: a linear phase term kept OUTSIDE the spline:
 *                           Psi_m(f) = spline_m(f) + 2 pi f t_shift, the same for every mode (reading R32)
 *   params                : [n_w][P], P = 5 + 2 n_c n_m:
 *                           Mc[s], q, t_c[s], phi_c[rad], 1/D, then T^c_m (re, im), m-major, c-minor
 *   A0, A1                : [n_c][n_b][2];  B0, B1 : [n_c][n_b];  h0_edges : [n_c][n_e][2]
 *   grid                  : f_k = (double)k * df, k = k_min + i
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef long double ld;

/* threads the walker loops run on (timing harness only: bench.py reports the oracle per core and on all cores) */
int orc_get_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
int orc_set_threads(int n)
{
#ifdef _OPENMP
    if (n >= 1) omp_set_num_threads(n);
#endif
    return orc_get_threads();
}

static const ld PI_L = 3.14159265358979323846264338327950288L;

/* ---------------------------------------------------------------------------------------------
 * Natural cubic spline (R1).  Unknowns M_j = y''(x_j):
 *   (h_{j-1}/6) M_{j-1} + ((h_{j-1}+h_j)/3) M_j + (h_j/6) M_{j+1}
 *        = (y_{j+1}-y_j)/h_j - (y_j-y_{j-1})/h_{j-1},   j = 1..n-2,   M_0 = M_{n-1} = 0.
 * Naive Thomas elimination.
 * ------------------------------------------------------------------------------------------- */
static int spline_natural_ld(int n, const double *x, const ld *y, ld *M)
{
    if (n < 3) return -1;
    ld *cp = (ld *)malloc(sizeof(ld) * (size_t)n);
    ld *dp = (ld *)malloc(sizeof(ld) * (size_t)n);
    if (!cp || !dp) { free(cp); free(dp); return -4; }
    M[0] = 0.0L; M[n - 1] = 0.0L;
    /* forward sweep over rows j = 1..n-2 */
    for (int j = 1; j <= n - 2; ++j) {
        ld hm = (ld)x[j] - (ld)x[j - 1];
        ld hp = (ld)x[j + 1] - (ld)x[j];
        ld a = hm / 6.0L;                 /* sub-diagonal   */
        ld b = (hm + hp) / 3.0L;          /* diagonal       */
        ld c = hp / 6.0L;                 /* super-diagonal */
        ld r = (y[j + 1] - y[j]) / hp - (y[j] - y[j - 1]) / hm;
        if (j == 1) {                     /* M_0 = 0 removes the sub-diagonal term */
            cp[j] = c / b;
            dp[j] = r / b;
        } else {
            ld den = b - a * cp[j - 1];
            cp[j] = c / den;
            dp[j] = (r - a * dp[j - 1]) / den;
        }
    }
    /* back substitution; M_{n-1} = 0 */
    for (int j = n - 2; j >= 1; --j)
        M[j] = dp[j] - cp[j] * M[j + 1];
    free(cp); free(dp);
    return 0;
}

/* ---------------------------------------------------------------------------------------------
 * Not-a-knot cubic spline (R1 lists it as the optional boundary condition).
 * The interior rows are those of the natural spline.  The two end conditions say that the third derivative is
 * continuous across x_1 and across x_{n-2}:
 *   (M_1 - M_0)/h_0 = (M_2 - M_1)/h_1              =>  M_0     = (1 + h_0/h_1) M_1 - (h_0/h_1) M_2
 *   (M_{n-1} - M_{n-2})/h_{n-2} = (M_{n-2} - M_{n-3})/h_{n-3}
 *                                                  =>  M_{n-1} = (1 + h_{n-2}/h_{n-3}) M_{n-2} - (h_{n-2}/h_{n-3}) M_{n-3}
 * Substituting them into rows 1 and n-2 keeps the system tridiagonal in M_1..M_{n-2} (n >= 4):
 *   row 1  : [ (h_0+h_1)/3 + (h_0/6)(1 + h_0/h_1) ] M_1 + [ h_1/6 - (h_0/6)(h_0/h_1) ] M_2 = r_1
 *   row n-2: [ h_{n-3}/6 - (h_{n-2}/6)(h_{n-2}/h_{n-3}) ] M_{n-3}
 *            + [ (h_{n-3}+h_{n-2})/3 + (h_{n-2}/6)(1 + h_{n-2}/h_{n-3}) ] M_{n-2} = r_{n-2}
 * Naive Thomas elimination, then the two end values.
 * ------------------------------------------------------------------------------------------- */
static int spline_notaknot_ld(int n, const double *x, const ld *y, ld *M)
{
    if (n < 4) return -1;
    ld *cp = (ld *)malloc(sizeof(ld) * (size_t)n);
    ld *dp = (ld *)malloc(sizeof(ld) * (size_t)n);
    if (!cp || !dp) { free(cp); free(dp); return -4; }
    const ld h0 = (ld)x[1] - (ld)x[0], h1 = (ld)x[2] - (ld)x[1];
    const ld hl = (ld)x[n - 1] - (ld)x[n - 2], hk = (ld)x[n - 2] - (ld)x[n - 3];
    const ld rho0 = h0 / h1, rhon = hl / hk;
    for (int j = 1; j <= n - 2; ++j) {
        ld hm = (ld)x[j] - (ld)x[j - 1];
        ld hp = (ld)x[j + 1] - (ld)x[j];
        ld a = hm / 6.0L, b = (hm + hp) / 3.0L, c = hp / 6.0L;
        ld r = (y[j + 1] - y[j]) / hp - (y[j] - y[j - 1]) / hm;
        if (j == 1)     { b += a * (1.0L + rho0); c -= a * rho0; a = 0.0L; }
        if (j == n - 2) { b += c * (1.0L + rhon); a -= c * rhon; c = 0.0L; }
        if (j == 1) {
            cp[j] = c / b;
            dp[j] = r / b;
        } else {
            ld den = b - a * cp[j - 1];
            cp[j] = c / den;
            dp[j] = (r - a * dp[j - 1]) / den;
        }
    }
    M[n - 2] = dp[n - 2];
    for (int j = n - 3; j >= 1; --j)
        M[j] = dp[j] - cp[j] * M[j + 1];
    M[0] = (1.0L + rho0) * M[1] - rho0 * M[2];
    M[n - 1] = (1.0L + rhon) * M[n - 2] - rhon * M[n - 3];
    free(cp); free(dp);
    return 0;
}

/* Which boundary condition the splines of this library use: 0 natural (the default, reading R1), 1 not-a-knot.
 * One process-wide switch (set it before a call, not during one), so that every path that splines node arrays
 * (amplitude, phase, transfer function) follows it without a second copy of each entry point. */
static int g_spline_bc = 0;
int orc_set_spline_bc(int bc)
{
    if (bc != 0 && bc != 1) return -1;
    g_spline_bc = bc;
    return 0;
}
static int spline_ld(int n, const double *x, const ld *y, ld *M)
{
    return g_spline_bc ? spline_notaknot_ld(n, x, y, M) : spline_natural_ld(n, x, y, M);
}

/* interval index: largest j with x_j <= f, clamped to [0, n-2] (R21) */
static int find_interval(int n, const double *x, double f)
{
    int j = 0;
    while (j < n - 2 && x[j + 1] <= f) ++j;   /* plain linear search */
    return j;
}

/* y(f) on [x_j, x_{j+1}], t = f - x_j:
 *   y = y_j + b_j t + (M_j/2) t^2 + ((M_{j+1}-M_j)/(6 h_j)) t^3,
 *   b_j = (y_{j+1}-y_j)/h_j - h_j (2 M_j + M_{j+1})/6 */
static ld spline_eval_ld(const double *x, const ld *y, const ld *M, int j, double f)
{
    ld h = (ld)x[j + 1] - (ld)x[j];
    ld t = (ld)f - (ld)x[j];
    ld b = (y[j + 1] - y[j]) / h - h * (2.0L * M[j] + M[j + 1]) / 6.0L;
    ld c = M[j] / 2.0L;
    ld dd = (M[j + 1] - M[j]) / (6.0L * h);
    return y[j] + b * t + c * t * t + dd * t * t * t;
}

/* exported for pins: second derivatives and point evaluation in one call */
int orc_spline_natural(int n, const double *x, const double *y, double *M_out)
{
    ld *yl = (ld *)malloc(sizeof(ld) * (size_t)n), *M = (ld *)malloc(sizeof(ld) * (size_t)n);
    if (!yl || !M) { free(yl); free(M); return -4; }
    for (int j = 0; j < n; ++j) yl[j] = (ld)y[j];
    int rc = spline_natural_ld(n, x, yl, M);
    if (rc == 0) for (int j = 0; j < n; ++j) M_out[j] = (double)M[j];
    free(yl); free(M);
    return rc;
}

int orc_spline_second_derivatives(int n, const double *x, const double *y, double *M_out)
{
    ld *yl = (ld *)malloc(sizeof(ld) * (size_t)n), *M = (ld *)malloc(sizeof(ld) * (size_t)n);
    if (!yl || !M) { free(yl); free(M); return -4; }
    for (int j = 0; j < n; ++j) yl[j] = (ld)y[j];
    int rc = spline_ld(n, x, yl, M);
    if (rc == 0) for (int j = 0; j < n; ++j) M_out[j] = (double)M[j];
    free(yl); free(M);
    return rc;
}

int orc_spline_eval(int n, const double *x, const double *y, int64_t n_q, const double *f_q, double *out)
{
    ld *yl = (ld *)malloc(sizeof(ld) * (size_t)n), *M = (ld *)malloc(sizeof(ld) * (size_t)n);
    if (!yl || !M) { free(yl); free(M); return -4; }
    for (int j = 0; j < n; ++j) yl[j] = (ld)y[j];
    int rc = spline_ld(n, x, yl, M);
    if (rc == 0)
        for (int64_t i = 0; i < n_q; ++i)
            out[i] = (double)spline_eval_ld(x, yl, M, find_interval(n, x, f_q[i]), f_q[i]);
    free(yl); free(M);
    return rc;
}

/* ---------------------------------------------------------------------------------------------
 * TaylorF2 stand-in waveform (BASELINE.json configs 0 and 3; NOT from PAPER.md; R9).
 *   M = Mc eta^(-3/5), eta = q/(1+q)^2, v = (pi M f)^(1/3), f_ISCO = 6^(-3/2)/(pi M)
 *   Psi(f)   = 2 pi f t_c - phi_c - pi/4 + 3/(128 eta v^5)
 *   A_lm(f)  = c_lm f^(-7/6)/D * taper(2f/(m f_ISCO))
 *   Psi_lm(f)= (m/2) Psi(2f/m)
 *   taper(x) = 1 (x<=1); s^3(10-15s+6s^2), s=(1+kappa-x)/kappa (1<x<1+kappa); 0 beyond.
 * ------------------------------------------------------------------------------------------- */
static ld taper_l(ld x, ld kappa)
{
    if (x <= 1.0L) return 1.0L;
    if (x >= 1.0L + kappa) return 0.0L;
    ld s = (1.0L + kappa - x) / kappa;
    return s * s * s * (10.0L - 15.0L * s + 6.0L * s * s);
}

static ld psi22_l(ld f, ld Mtot, ld eta, ld t_c, ld phi_c)
{
    ld v = cbrtl(PI_L * Mtot * f);
    ld v5 = v * v * v * v * v;
    return 2.0L * PI_L * f * t_c - phi_c - PI_L / 4.0L + 3.0L / (128.0L * eta * v5);
}

static void standin_masses(const double *p, ld *Mtot, ld *eta, ld *f_isco)
{
    ld Mc = (ld)p[0], q = (ld)p[1];
    *eta = q / ((1.0L + q) * (1.0L + q));
    *Mtot = Mc * powl(*eta, -0.6L);
    *f_isco = powl(6.0L, -1.5L) / (PI_L * (*Mtot));
}

/* amplitude and phase (radians) of mode (l,m) at frequency f for parameter row p.  split_tc: the phase WITHOUT its
 * linear term 2 pi f t_c ((m/2) 2 pi (2f/m) t_c = 2 pi f t_c for every mode), which then travels as t_shift = t_c */
static void standin_mode(const double *p, int m, double c_lm, double kappa, double f, int split_tc, ld *amp, ld *phase)
{
    ld Mtot, eta, f_isco;
    standin_masses(p, &Mtot, &eta, &f_isco);
    ld t_c = split_tc ? 0.0L : (ld)p[2], phi_c = (ld)p[3], invD = (ld)p[4];
    ld fl = (ld)f, mh = (ld)m / 2.0L;
    *amp = (ld)c_lm * powl(fl, -7.0L / 6.0L) * invD * taper_l(2.0L * fl / ((ld)m * f_isco), (ld)kappa);
    *phase = mh * psi22_l(fl / mh, Mtot, eta, t_c, phi_c);
}

int orc_standin_fisco(const double *p, double *f_isco_out)
{
    ld Mtot, eta, fi;
    standin_masses(p, &Mtot, &eta, &fi);
    *f_isco_out = (double)fi;
    return 0;
}

/* node arrays for a batch: amp, phase [n_w][n_m][n_freq] (rounded to fp64: they are the arrays the
 * array entry point would be given), tf [n_w][n_m][n_c][2], band [n_w][2] (R10):
 * band = [k_min df, min(k_max df, (1+kappa) f_ISCO max_m(m/2))]. */
int orc_standin_nodes(int64_t n_w, int n_m, int n_c, const int32_t *mode_m, const double *c_lm, double kappa,
                      const double *params, int n_freq, const double *f,
                      double f_grid_lo, double f_grid_hi, int split_tc,
                      double *amp, double *phase, double *tf, double *band)
{
    const int P = 5 + 2 * n_c * n_m;
    int m_max = 0;
    for (int im = 0; im < n_m; ++im) if (mode_m[im] > m_max) m_max = mode_m[im];
    #pragma omp parallel for schedule(static)
    for (int64_t w = 0; w < n_w; ++w) {
        const double *p = params + w * P;
        for (int im = 0; im < n_m; ++im)
            for (int j = 0; j < n_freq; ++j) {
                ld a, ph;
                standin_mode(p, mode_m[im], c_lm[im], kappa, f[j], split_tc, &a, &ph);
                amp[(w * n_m + im) * n_freq + j] = (double)a;
                phase[(w * n_m + im) * n_freq + j] = (double)ph;
            }
        if (tf) memcpy(tf + w * n_m * n_c * 2, p + 5, sizeof(double) * (size_t)(n_m * n_c * 2));
        if (band) {
            ld Mtot, eta, fi;
            standin_masses(p, &Mtot, &eta, &fi);
            ld top = (1.0L + (ld)kappa) * fi * ((ld)m_max / 2.0L);
            band[2 * w] = f_grid_lo;
            band[2 * w + 1] = (top < (ld)f_grid_hi) ? (double)top : f_grid_hi;
        }
    }
    return 0;
}

/* ---------------------------------------------------------------------------------------------
 * <d|d> = sum_c sum_k W_k |d^c_k|^2     (Eq. 3 with W_k = 4 df w_k / S_n)
 * ------------------------------------------------------------------------------------------- */
/* weight of channel c at bin i: one row shared by all channels (w_rows = 1) or one row per channel */
static ld wgt(const double *W, int w_rows, int64_t n_f, int c, int64_t i)
{
    return (ld)W[(w_rows > 1 ? (int64_t)c * n_f : 0) + i];
}

static ld inner_dd(int n_c, int64_t n_f, const double *d, const double *W, int w_rows, int64_t i_lo, int64_t i_hi)
{
    ld s = 0.0L;
    for (int c = 0; c < n_c; ++c)
        for (int64_t i = i_lo; i < i_hi; ++i) {
            ld re = d[(c * n_f + i) * 2], im = d[(c * n_f + i) * 2 + 1];
            s += wgt(W, w_rows, n_f, c, i) * (re * re + im * im);
        }
    return s;
}

int orc_inner(int n_c, int64_t n_f, const double *a, const double *b, const double *W, int w_rows, double *re_out,
              double *im_out)
{
    if (w_rows != 1 && w_rows != n_c) return -1;
    /* sum_c sum_k W_k conj(a_k) b_k : real part is <a|b> */
    ld sr = 0.0L, si = 0.0L;
    for (int c = 0; c < n_c; ++c)
        for (int64_t i = 0; i < n_f; ++i) {
            ld ar = a[(c * n_f + i) * 2], ai = a[(c * n_f + i) * 2 + 1];
            ld br = b[(c * n_f + i) * 2], bi = b[(c * n_f + i) * 2 + 1];
            sr += wgt(W, w_rows, n_f, c, i) * (ar * br + ai * bi);
            si += wgt(W, w_rows, n_f, c, i) * (ar * bi - ai * br);
        }
    *re_out = (double)sr; *im_out = (double)si;
    return 0;
}

/* ---------------------------------------------------------------------------------------------
 * Full-grid path (steps F2-F4 of DESIGN.md; SURVEY.md §8(c) "Algorithm, full-grid").
 * Per walker: spline amp and phase of every mode; for each dense bin inside the band
 *   h^c_k = sum_m T^c_m A_m(f_k) (cos Psi_m(f_k) - i sin Psi_m(f_k));          Eq. 7, 9
 *   d_h = sum_c sum_k W_k Re[conj(d^c_k) h^c_k],  h_h = sum_c sum_k W_k |h^c_k|^2;   Eq. 3
 *   log L = d_h - h_h/2 - <d|d>/2;   also the direct form -1/2 sum W |d-h|^2.       Eq. 2
 * If h_out != NULL (n_w must be 1) the dense template [n_c][n_f][2] is written too.
 * ------------------------------------------------------------------------------------------- */
int orc_full_batch(int64_t n_w, int n_m, int n_c, int n_nodes, const double *f_nodes,
                   const double *amp, const double *phase, const double *tf, const double *band,
                   int64_t n_f, int64_t k_min, double df, const double *d, const double *W, int w_rows,
                   const double *t_shift,
                   double *logL, double *d_h, double *h_h, double *logL_direct, double *h_out)
{
    if (n_nodes < 3 || n_m < 1 || n_c < 1 || n_c > 3) return -1;
    if (w_rows != 1 && w_rows != n_c) return -1;
    if (h_out && n_w != 1) return -1;
    const ld dd = d ? inner_dd(n_c, n_f, d, W, w_rows, 0, n_f) : 0.0L;
    int fail = 0;
    #pragma omp parallel for schedule(dynamic, 1)
    for (int64_t w = 0; w < n_w; ++w) {
        const size_t nn = (size_t)n_nodes;
        ld *yA = (ld *)malloc(sizeof(ld) * nn * (size_t)n_m), *MA = (ld *)malloc(sizeof(ld) * nn * (size_t)n_m);
        ld *yP = (ld *)malloc(sizeof(ld) * nn * (size_t)n_m), *MP = (ld *)malloc(sizeof(ld) * nn * (size_t)n_m);
        if (!yA || !MA || !yP || !MP) { fail = 1; free(yA); free(MA); free(yP); free(MP); continue; }
        for (int m = 0; m < n_m; ++m) {
            for (int j = 0; j < n_nodes; ++j) {
                yA[m * nn + j] = (ld)amp[(w * n_m + m) * nn + j];
                yP[m * nn + j] = (ld)phase[(w * n_m + m) * nn + j];
            }
            spline_ld(n_nodes, f_nodes, yA + m * nn, MA + m * nn);
            spline_ld(n_nodes, f_nodes, yP + m * nn, MP + m * nn);
        }
        const double f_lo = band ? band[2 * w] : -HUGE_VAL, f_hi = band ? band[2 * w + 1] : HUGE_VAL;
        const ld tsh = t_shift ? (ld)t_shift[w] : 0.0L;
        ld s_dh = 0.0L, s_hh = 0.0L, s_res = 0.0L;
        for (int c = 0; c < n_c; ++c)
            for (int64_t i = 0; i < n_f; ++i) {
                const double f = (double)(k_min + i) * df;
                const ld Wi = wgt(W, w_rows, n_f, c, i);
                ld hr = 0.0L, hi = 0.0L;
                if (f >= f_lo && f <= f_hi) {
                    const int j = find_interval(n_nodes, f_nodes, f);
                    for (int m = 0; m < n_m; ++m) {
                        ld A = spline_eval_ld(f_nodes, yA + m * nn, MA + m * nn, j, f);
                        ld Psi = spline_eval_ld(f_nodes, yP + m * nn, MP + m * nn, j, f);
                        if (t_shift) Psi += 2.0L * PI_L * (ld)f * tsh;        /* linear term outside the spline (R32) */
                        ld mr = A * cosl(Psi), mi = -A * sinl(Psi);          /* Eq. 7: A e^{-i Psi} */
                        ld tr = tf[((w * n_m + m) * n_c + c) * 2], ti = tf[((w * n_m + m) * n_c + c) * 2 + 1];
                        hr += tr * mr - ti * mi;                             /* Eq. 9 */
                        hi += tr * mi + ti * mr;
                    }
                }
                if (h_out) { h_out[(c * n_f + i) * 2] = (double)hr; h_out[(c * n_f + i) * 2 + 1] = (double)hi; }
                if (d) {
                    ld dr = d[(c * n_f + i) * 2], di = d[(c * n_f + i) * 2 + 1];
                    s_dh += Wi * (dr * hr + di * hi);                        /* Re[conj(d) h] */
                    s_res += Wi * ((dr - hr) * (dr - hr) + (di - hi) * (di - hi));
                }
                s_hh += Wi * (hr * hr + hi * hi);
            }
        if (logL) logL[w] = (double)(s_dh - 0.5L * s_hh - 0.5L * dd);
        if (d_h) d_h[w] = (double)s_dh;
        if (h_h) h_h[w] = (double)s_hh;
        if (logL_direct) logL_direct[w] = (double)(-0.5L * s_res);
        free(yA); free(MA); free(yP); free(MP);
    }
    return fail ? -4 : 0;
}

/* ---------------------------------------------------------------------------------------------
 * Full-grid path with a frequency-dependent transfer function.
 *   h~^{A,E}(f) = sum_lm T^{A,E}(f, t_lm(f)) h~_lm(f)                          Eq. 9
 * The transfer function's formula is in the paper's ref. [44], not in PAPER.md, so T arrives as caller
 * arrays at the spline nodes, T_nodes [n_w][n_m][n_c][n_nodes][2] (re, im); its real and imaginary parts
 * are splined exactly like amplitude and phase (natural cubic in f, reading R1) and evaluated per bin.
 * Everything else is orc_full_batch.
 * ------------------------------------------------------------------------------------------- */
int orc_full_batch_tf(int64_t n_w, int n_m, int n_c, int n_nodes, const double *f_nodes,
                      const double *amp, const double *phase, const double *tf_nodes, const double *band,
                      int64_t n_f, int64_t k_min, double df, const double *d, const double *W, int w_rows,
                      const double *t_shift,
                      double *logL, double *d_h, double *h_h, double *logL_direct, double *h_out)
{
    if (n_nodes < 3 || n_m < 1 || n_c < 1 || n_c > 3) return -1;
    if (w_rows != 1 && w_rows != n_c) return -1;
    if (h_out && n_w != 1) return -1;
    const ld dd = d ? inner_dd(n_c, n_f, d, W, w_rows, 0, n_f) : 0.0L;
    int fail = 0;
    #pragma omp parallel for schedule(dynamic, 1)
    for (int64_t w = 0; w < n_w; ++w) {
        const size_t nn = (size_t)n_nodes;
        const size_t ns = (size_t)n_m * (2 + 2 * (size_t)n_c);      /* splines per walker */
        ld *y = (ld *)malloc(sizeof(ld) * nn * ns), *M = (ld *)malloc(sizeof(ld) * nn * ns);
        if (!y || !M) { fail = 1; free(y); free(M); continue; }
        /* spline s of mode m: 0 amplitude, 1 phase, 2 + 2c Re T^c, 3 + 2c Im T^c */
        for (int m = 0; m < n_m; ++m) {
            ld *ym = y + (size_t)m * (2 + 2 * n_c) * nn, *Mm = M + (size_t)m * (2 + 2 * n_c) * nn;
            for (int j = 0; j < n_nodes; ++j) {
                ym[0 * nn + j] = (ld)amp[(w * n_m + m) * nn + j];
                ym[1 * nn + j] = (ld)phase[(w * n_m + m) * nn + j];
                for (int c = 0; c < n_c; ++c) {
                    const double *t = tf_nodes + ((((size_t)w * n_m + m) * n_c + c) * nn + j) * 2;
                    ym[(2 + 2 * c) * nn + j] = (ld)t[0];
                    ym[(3 + 2 * c) * nn + j] = (ld)t[1];
                }
            }
            for (int s = 0; s < 2 + 2 * n_c; ++s) spline_ld(n_nodes, f_nodes, ym + s * nn, Mm + s * nn);
        }
        const double f_lo = band ? band[2 * w] : -HUGE_VAL, f_hi = band ? band[2 * w + 1] : HUGE_VAL;
        const ld tsh = t_shift ? (ld)t_shift[w] : 0.0L;
        ld s_dh = 0.0L, s_hh = 0.0L, s_res = 0.0L;
        for (int c = 0; c < n_c; ++c)
            for (int64_t i = 0; i < n_f; ++i) {
                const double f = (double)(k_min + i) * df;
                const ld Wi = wgt(W, w_rows, n_f, c, i);
                ld hr = 0.0L, hi = 0.0L;
                if (f >= f_lo && f <= f_hi) {
                    const int j = find_interval(n_nodes, f_nodes, f);
                    for (int m = 0; m < n_m; ++m) {
                        const ld *ym = y + (size_t)m * (2 + 2 * n_c) * nn, *Mm = M + (size_t)m * (2 + 2 * n_c) * nn;
                        ld A = spline_eval_ld(f_nodes, ym, Mm, j, f);
                        ld Psi = spline_eval_ld(f_nodes, ym + nn, Mm + nn, j, f);
                        ld tr = spline_eval_ld(f_nodes, ym + (2 + 2 * c) * nn, Mm + (2 + 2 * c) * nn, j, f);
                        ld ti = spline_eval_ld(f_nodes, ym + (3 + 2 * c) * nn, Mm + (3 + 2 * c) * nn, j, f);
                        if (t_shift) Psi += 2.0L * PI_L * (ld)f * tsh;        /* linear term outside the spline (R32) */
                        ld mr = A * cosl(Psi), mi = -A * sinl(Psi);          /* Eq. 7: A e^{-i Psi} */
                        hr += tr * mr - ti * mi;                             /* Eq. 9 */
                        hi += tr * mi + ti * mr;
                    }
                }
                if (h_out) { h_out[(c * n_f + i) * 2] = (double)hr; h_out[(c * n_f + i) * 2 + 1] = (double)hi; }
                if (d) {
                    ld dr = d[(c * n_f + i) * 2], di = d[(c * n_f + i) * 2 + 1];
                    s_dh += Wi * (dr * hr + di * hi);
                    s_res += Wi * ((dr - hr) * (dr - hr) + (di - hi) * (di - hi));
                }
                s_hh += Wi * (hr * hr + hi * hi);
            }
        if (logL) logL[w] = (double)(s_dh - 0.5L * s_hh - 0.5L * dd);
        if (d_h) d_h[w] = (double)s_dh;
        if (h_h) h_h[w] = (double)s_hh;
        if (logL_direct) logL_direct[w] = (double)(-0.5L * s_res);
        free(y); free(M);
    }
    return fail ? -4 : 0;
}

/* ---------------------------------------------------------------------------------------------
 * Time-frequency correspondence at the spline nodes                              Eq. 8
 *   t_lm(f) = t_ref - (1/2pi) d phi_lm / df
 * with d phi/df the first derivative of the natural cubic spline of the node phases (reading R1):
 *   y'(x_j)     = (y_{j+1}-y_j)/h_j - h_j (2 M_j + M_{j+1})/6          j < n-1  (left end of interval j)
 *   y'(x_{n-1}) = (y_{n-1}-y_{n-2})/h + h (M_{n-2} + 2 M_{n-1})/6      (right end of the last interval)
 * phase [n_w][n_m][n_nodes] radians -> t_lm [n_w][n_m][n_nodes] seconds.
 * ------------------------------------------------------------------------------------------- */
int orc_tlm_nodes(int64_t n_w, int n_m, int n_nodes, const double *f_nodes, const double *phase, double t_ref,
                  double *t_lm)
{
    if (n_nodes < 3 || n_m < 1) return -1;
    int fail = 0;
    #pragma omp parallel for schedule(static)
    for (int64_t s = 0; s < n_w * n_m; ++s) {
        const size_t nn = (size_t)n_nodes;
        ld *y = (ld *)malloc(sizeof(ld) * nn), *M = (ld *)malloc(sizeof(ld) * nn);
        if (!y || !M) { fail = 1; free(y); free(M); continue; }
        for (int j = 0; j < n_nodes; ++j) y[j] = (ld)phase[(size_t)s * nn + j];
        spline_natural_ld(n_nodes, f_nodes, y, M);
        for (int j = 0; j < n_nodes; ++j) {
            ld dy;
            if (j < n_nodes - 1) {
                const ld h = (ld)f_nodes[j + 1] - (ld)f_nodes[j];
                dy = (y[j + 1] - y[j]) / h - h * (2.0L * M[j] + M[j + 1]) / 6.0L;
            } else {
                const ld h = (ld)f_nodes[j] - (ld)f_nodes[j - 1];
                dy = (y[j] - y[j - 1]) / h + h * (M[j - 1] + 2.0L * M[j]) / 6.0L;
            }
            t_lm[(size_t)s * nn + j] = (double)((ld)t_ref - dy / (2.0L * PI_L));
        }
        free(y); free(M);
    }
    return fail ? -4 : 0;
}

int orc_dd(int n_c, int64_t n_f, const double *d, const double *W, int w_rows, double *dd_out)
{
    if (w_rows != 1 && w_rows != n_c) return -1;
    *dd_out = (double)inner_dd(n_c, n_f, d, W, w_rows, 0, n_f);
    return 0;
}

/* stand-in template evaluated DIRECTLY (no spline) at arbitrary frequencies: h [n_c][n_freq][2].
 * Used for the het reference h0 (dense grid and edges, R12) and inside orc_het_batch_standin.
 * Outside [f_lo, f_hi] the template is zero (band mask, R10). */
int orc_standin_direct(int n_m, int n_c, const int32_t *mode_m, const double *c_lm, double kappa,
                       const double *p, int64_t n_freq, const double *f, double f_lo, double f_hi, double *h)
{
    #pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n_freq; ++i) {
        for (int c = 0; c < n_c; ++c) {
            ld hr = 0.0L, hi = 0.0L;
            if (f[i] >= f_lo && f[i] <= f_hi)
                for (int m = 0; m < n_m; ++m) {
                    ld A, Psi;
                    standin_mode(p, mode_m[m], c_lm[m], kappa, f[i], 0, &A, &Psi);
                    ld mr = A * cosl(Psi), mi = -A * sinl(Psi);
                    ld tr = p[5 + (m * n_c + c) * 2], ti = p[5 + (m * n_c + c) * 2 + 1];
                    hr += tr * mr - ti * mi;
                    hi += tr * mi + ti * mr;
                }
            h[(c * n_freq + i) * 2] = (double)hr;
            h[(c * n_freq + i) * 2 + 1] = (double)hi;
        }
    }
    return 0;
}

/* ---------------------------------------------------------------------------------------------
 * Heterodyne summary data (step H0; Eq. 15, 16, 18, 19 with 4 Delta f folded into W_k).
 * Bin b = [e_b, e_{b+1}) (last bin closed), f_b = (e_b + e_{b+1})/2 (R13):
 *   A0 = sum W d conj(h0),  A1 = sum W d conj(h0) (f - f_b),
 *   B0 = sum W |h0|^2,      B1 = sum W |h0|^2 (f - f_b),     dd_band = sum_c sum_{k in any bin} W |d|^2.
 * B2 = sum W |h0|^2 (f-f_b)^2 is returned for the pin on the term Eq. 17 drops (may be NULL).
 * ------------------------------------------------------------------------------------------- */
int orc_het_prepare(int n_c, int64_t n_f, int64_t k_min, double df, const double *d, const double *W, int w_rows,
                    const double *h0, int n_e, const double *e,
                    double *A0, double *A1, double *B0, double *B1, double *B2, double *dd_band)
{
    if (n_e < 2) return -1;
    if (w_rows != 1 && w_rows != n_c) return -1;
    const int n_b = n_e - 1;
    ld ddb = 0.0L;
    for (int c = 0; c < n_c; ++c)
        for (int b = 0; b < n_b; ++b) {
            const ld fb = 0.5L * ((ld)e[b] + (ld)e[b + 1]);
            ld a0r = 0, a0i = 0, a1r = 0, a1i = 0, b0 = 0, b1 = 0, b2 = 0;
            for (int64_t i = 0; i < n_f; ++i) {
                const double f = (double)(k_min + i) * df;
                const int inside = (f >= e[b]) && (b == n_b - 1 ? f <= e[b + 1] : f < e[b + 1]);
                if (!inside) continue;
                ld dr = d[(c * n_f + i) * 2], di = d[(c * n_f + i) * 2 + 1];
                ld hr = h0[(c * n_f + i) * 2], hi = h0[(c * n_f + i) * 2 + 1];
                ld w = wgt(W, w_rows, n_f, c, i), t = (ld)f - fb;
                ld pr = dr * hr + di * hi, pi = di * hr - dr * hi;     /* d conj(h0) */
                ld h2 = hr * hr + hi * hi;
                a0r += w * pr;      a0i += w * pi;
                a1r += w * pr * t;  a1i += w * pi * t;
                b0 += w * h2;  b1 += w * h2 * t;  b2 += w * h2 * t * t;
                ddb += w * (dr * dr + di * di);
            }
            A0[(c * n_b + b) * 2] = (double)a0r; A0[(c * n_b + b) * 2 + 1] = (double)a0i;
            A1[(c * n_b + b) * 2] = (double)a1r; A1[(c * n_b + b) * 2 + 1] = (double)a1i;
            B0[c * n_b + b] = (double)b0; B1[c * n_b + b] = (double)b1;
            if (B2) B2[c * n_b + b] = (double)b2;
        }
    *dd_band = (double)ddb;
    return 0;
}

/* ---------------------------------------------------------------------------------------------
 * Heterodyned likelihood (steps H1-H3).  amp_e, phase_e [n_w][n_m][n_e] at the bin edges.
 *   h^c(e) = sum_m T^c_m A_m e^{-i Psi_m};  r^c(e) = h^c(e)/h0^c(e);
 *   r0 = (r_lo + r_hi)/2,  r1 = (r_hi - r_lo)/(e_{b+1} - e_b);                       Eq. 11
 *   d_h = sum_c sum_b Re[A0 conj(r0) + A1 conj(r1)];                                 Eq. 14
 *   h_h = sum_c sum_b B0 |r0|^2 + 2 B1 Re[r0 conj(r1)];                              Eq. 17
 *   log L = d_h - h_h/2 - dd_band/2.                                                 Eq. 2
 * Returns -6 if h0 is exactly zero (or non-finite) at an edge.
 * ------------------------------------------------------------------------------------------- */
int orc_het_batch(int64_t n_w, int n_m, int n_c, int n_e, const double *e,
                  const double *amp_e, const double *phase_e, const double *tf, const double *t_shift, const double *h0_e,
                  const double *A0, const double *A1, const double *B0, const double *B1, double dd_band,
                  double *logL, double *d_h, double *h_h)
{
    if (n_e < 2) return -1;
    const int n_b = n_e - 1;
    for (int c = 0; c < n_c; ++c)
        for (int j = 0; j < n_e; ++j) {
            double m2 = h0_e[(c * n_e + j) * 2] * h0_e[(c * n_e + j) * 2] + h0_e[(c * n_e + j) * 2 + 1] * h0_e[(c * n_e + j) * 2 + 1];
            if (!(m2 > 0.0) || !isfinite(m2)) return -6;
        }
    int fail = 0;
    #pragma omp parallel for schedule(static)
    for (int64_t w = 0; w < n_w; ++w) {
        ld *rr = (ld *)malloc(sizeof(ld) * (size_t)n_e), *ri = (ld *)malloc(sizeof(ld) * (size_t)n_e);
        if (!rr || !ri) { fail = 1; free(rr); free(ri); continue; }
        ld s_dh = 0.0L, s_hh = 0.0L;
        for (int c = 0; c < n_c; ++c) {
            for (int j = 0; j < n_e; ++j) {
                ld hr = 0.0L, hi = 0.0L;
                for (int m = 0; m < n_m; ++m) {
                    ld A = amp_e[(w * n_m + m) * n_e + j], Psi = phase_e[(w * n_m + m) * n_e + j];
                    if (t_shift) Psi += 2.0L * PI_L * (ld)e[j] * (ld)t_shift[w];  /* linear term kept apart (R32) */
                    ld mr = A * cosl(Psi), mi = -A * sinl(Psi);
                    ld tr = tf[((w * n_m + m) * n_c + c) * 2], ti = tf[((w * n_m + m) * n_c + c) * 2 + 1];
                    hr += tr * mr - ti * mi;
                    hi += tr * mi + ti * mr;
                }
                ld gr = h0_e[(c * n_e + j) * 2], gi = h0_e[(c * n_e + j) * 2 + 1];
                ld den = gr * gr + gi * gi;
                rr[j] = (hr * gr + hi * gi) / den;            /* h / h0 */
                ri[j] = (hi * gr - hr * gi) / den;
            }
            for (int b = 0; b < n_b; ++b) {
                ld r0r = 0.5L * (rr[b] + rr[b + 1]), r0i = 0.5L * (ri[b] + ri[b + 1]);
                ld wdt = (ld)e[b + 1] - (ld)e[b];
                ld r1r = (rr[b + 1] - rr[b]) / wdt, r1i = (ri[b + 1] - ri[b]) / wdt;
                ld a0r = A0[(c * n_b + b) * 2], a0i = A0[(c * n_b + b) * 2 + 1];
                ld a1r = A1[(c * n_b + b) * 2], a1i = A1[(c * n_b + b) * 2 + 1];
                s_dh += (a0r * r0r + a0i * r0i) + (a1r * r1r + a1i * r1i);     /* Re[A conj(r)] */
                s_hh += (ld)B0[c * n_b + b] * (r0r * r0r + r0i * r0i)
                      + 2.0L * (ld)B1[c * n_b + b] * (r0r * r1r + r0i * r1i);
            }
        }
        if (logL) logL[w] = (double)(s_dh - 0.5L * s_hh - 0.5L * (ld)dd_band);
        if (d_h) d_h[w] = (double)s_dh;
        if (h_h) h_h[w] = (double)s_hh;
        free(rr); free(ri);
    }
    return fail ? -4 : 0;
}
