/*
 * oracle/lsp_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, fp64 CPU implementation of the Lomb-Scargle periodogram exactly as
 * the paper DEFINES it: the two-pass form, eq. (1) with the time offset tau of
 * eq. (2)  (section 3).  It is the yardstick the CUDA path in
 * paper_1007_1658_b200/csrc is compared against; it shares no code, header, table
 * or helper with that path and is never called by it.  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * build or call this file.
 *
 * No blocking, no recurrences, no refactoring (the single-pass form, eqs 5-8, is the
 * GPU's formulation and deliberately NOT used here): for every trial frequency
 *   1.  S2 = sum_j sin(2 w t_j),  C2 = sum_j cos(2 w t_j)           eq. (2)
 *   2.  tau = atan2(S2, C2) / (2 w)                                  eq. (2), reading G5
 *   3.  the four sums of eq. (1) with libm sin/cos of w (t_j - tau)
 *   4.  P = ( XC^2/CC + XS^2/SS ) / (2 var)                          eq. (1), readings G1, G7
 * with plain left-to-right fp64 accumulation.
 *
 * Readings of the paper where it is silent (DESIGN.md section "Readings"):
 *   G1  the series is "scaled and shifted" to zero mean and unit variance
 *       (PAPER.md:41): mean = sum x / Nt, var = sum (x-mean)^2 / (Nt-1)  (sample variance).
 *   G2  grid f_k = f_min + k*df evaluated as f_min + (double)k*df (PAPER.md:108 generalised).
 *   G5  tau is defined modulo pi/(2w); any branch gives the same P.  atan2(0,0) = 0.
 *   G6  no time shift is applied here (the CUDA path shifts by t[0]; P is invariant).
 *   G7  a term whose denominator is <= 1e-12*Nt is dropped (its numerator is 0 too);
 *       this makes P(f=0) = 0.
 *
 * Parity pins (tests/test_oracle_pins.py): brute-force least squares, FFT periodogram on
 * even sampling, time-shift invariance, closed form (Nt-1)/2, scipy.signal.lombscargle,
 * Gaussian-noise statistics, injected sinusoid, eqs (5)-(8) equivalence, mpmath brute force;
 * generalised periodogram GP1-GP6, weighted generalised periodogram GW1-GW5.
 */
#include <math.h>
#include <stdint.h>
#include <stddef.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define LSP_ORACLE_TWO_PI 6.283185307179586476925286766559

/* Mean and sample variance of x (fp32 input promoted to fp64), PAPER.md:41 + reading G1. */
void lsp_oracle_moments(const float* x, int64_t Nt, double* mean_out, double* var_out)
{
    double s = 0.0;
    for (int64_t j = 0; j < Nt; ++j) s += (double)x[j];
    double mean = s / (double)Nt;
    double q = 0.0;
    for (int64_t j = 0; j < Nt; ++j) {
        double d = (double)x[j] - mean;
        q += d * d;
    }
    *mean_out = mean;
    *var_out = q / (double)(Nt - 1);
}

/* One frequency, eqs (1)+(2).  X is the mean-subtracted series in fp64. */
static double lsp_oracle_one(const double* t, const double* X, int64_t Nt, double f, double var)
{
    const double w = LSP_ORACLE_TWO_PI * f;
    if (w == 0.0) {
        /* eq. (1) with w = 0: cos = 1, sin = 0; the sine term is 0/0 and dropped (G7). */
        double xc = 0.0;
        for (int64_t j = 0; j < Nt; ++j) xc += X[j];
        return (xc * xc / (double)Nt) / (2.0 * var);
    }
    double S2 = 0.0, C2 = 0.0;                       /* eq. (2) */
    for (int64_t j = 0; j < Nt; ++j) {
        double a = 2.0 * w * t[j];
        S2 += sin(a);
        C2 += cos(a);
    }
    const double tau = atan2(S2, C2) / (2.0 * w);    /* G5 */
    double XC = 0.0, XS = 0.0, CC = 0.0, SS = 0.0;   /* eq. (1) */
    for (int64_t j = 0; j < Nt; ++j) {
        double a = w * (t[j] - tau);
        double c = cos(a), s = sin(a);
        XC += X[j] * c;
        XS += X[j] * s;
        CC += c * c;
        SS += s * s;
    }
    const double eps = 1e-12 * (double)Nt;           /* G7 */
    double p = 0.0;
    if (CC > eps) p += XC * XC / CC;
    if (SS > eps) p += XS * XS / SS;
    return p / (2.0 * var);
}

/*
 * Periodogram of one series on selected grid points.
 *   t[Nt] fp64, x[Nt] fp32 (host), grid f_k = f_min + k*df.
 *   ks == NULL : evaluate k = 0..nk-1;  otherwise evaluate k = ks[i], i = 0..nk-1.
 *   P[nk] fp64 out.  scratch[Nt] fp64 (caller-provided, holds x - mean).
 *   nthreads <= 0 : use the OpenMP default.  Returns the number of threads used.
 */
int lsp_oracle_periodogram(const double* t, const float* x, int64_t Nt,
                           double f_min, double df, const int64_t* ks, int64_t nk,
                           double* P, double* scratch, int nthreads)
{
    double mean, var;
    lsp_oracle_moments(x, Nt, &mean, &var);
    for (int64_t j = 0; j < Nt; ++j) scratch[j] = (double)x[j] - mean;
    int used = 1;
#ifdef _OPENMP
    if (nthreads > 0) omp_set_num_threads(nthreads);
    #pragma omp parallel
    {
        #pragma omp single
        used = omp_get_num_threads();
    }
    #pragma omp parallel for schedule(dynamic, 4)
#endif
    for (int64_t i = 0; i < nk; ++i) {
        int64_t k = ks ? ks[i] : i;
        double f = f_min + (double)k * df;           /* G2 */
        P[i] = lsp_oracle_one(t, scratch, Nt, f, var);
    }
    return used;
}

/*
 * The least-squares fit both generalised periodograms below are defined by: for one frequency, minimise
 *     chi^2 = sum_j w_j (X_j - a cos(w t_j) - b sin(w t_j) - c)^2          (w_j = 1 when wts is NULL)
 * and return chi0^2 - chi^2_min, where X has zero (weighted) mean so that chi0^2 = sum_j w_j X_j^2 belongs to the constant
 * model.  Normal equations of three basis functions, Gaussian elimination with partial pivoting.
 *
 * Reading G15: the model space {cos, sin, 1} does not depend on the time origin or on which basis spans
 * it, so the fit is posed in the best-conditioned equivalent basis: times measured from their weighted mean,
 *     g0 = (cos(w t') - 1) - its weighted mean,   g1 = sin(w t') - its weighted mean,   g2 = 1,
 * with cos - 1 = -2 sin^2(w t'/2) formed without cancellation, and every basis function scaled to unit norm before the
 * elimination.  The chi^2 reduction is the same number (pin GP6: 60-digit arithmetic on the raw basis); what changes is that
 * it stays accurate as f T -> 0, where cos -> 1 runs into the constant and the raw normal equations lose every digit (the
 * earlier form of this function returned 0 below f T ~ 1e-3; the exact fit there is that of a constant + linear + quadratic
 * trend, which is not small for a series with a drift).  A fit that is singular even so -- a basis function that vanishes on
 * the samples (f = 0; the aliases of regular sampling), or two that coincide to 1e-12 -- returns 0 (reading G7 carried over).
 */
static double lsp_oracle_gls_fit(const double* t, const double* X, const double* wts, int64_t Nt, double f)
{
    const double om = LSP_ORACLE_TWO_PI * f;
    double wsum = 0.0, tbar = 0.0;
    for (int64_t j = 0; j < Nt; ++j) { const double w = wts ? wts[j] : 1.0; wsum += w; tbar += w * t[j]; }
    tbar /= wsum;
    double cbar = 0.0, sbar = 0.0;                                     /* weighted means of cos - 1 and sin */
    for (int64_t j = 0; j < Nt; ++j) {
        const double w = wts ? wts[j] : 1.0, a = om * (t[j] - tbar), sh = sin(0.5 * a);
        cbar += w * (-2.0 * sh * sh);
        sbar += w * sin(a);
    }
    cbar /= wsum; sbar /= wsum;
    double M[3][4] = {{0, 0, 0, 0}, {0, 0, 0, 0}, {0, 0, 0, 0}};      /* [A^T W A | A^T W X] */
    for (int64_t j = 0; j < Nt; ++j) {
        const double w = wts ? wts[j] : 1.0, a = om * (t[j] - tbar), sh = sin(0.5 * a);
        const double g[3] = {-2.0 * sh * sh - cbar, sin(a) - sbar, 1.0};
        for (int r = 0; r < 3; ++r) {
            for (int c = 0; c < 3; ++c) M[r][c] += w * g[r] * g[c];
            M[r][3] += w * g[r] * X[j];
        }
    }
    double norm[3];
    for (int r = 0; r < 3; ++r) {
        if (!(M[r][r] > 0.0)) return 0.0;                              /* a basis function that vanishes on the samples: G7 */
        norm[r] = sqrt(M[r][r]);
    }
    for (int r = 0; r < 3; ++r) {
        for (int c = 0; c < 3; ++c) M[r][c] /= norm[r] * norm[c];
        M[r][3] /= norm[r];
    }
    const double rhs[3] = {M[0][3], M[1][3], M[2][3]};
    const double tiny = 1e-12;                                         /* relative: the matrix now has a unit diagonal */
    for (int col = 0; col < 3; ++col) {                                /* elimination, partial pivoting */
        int piv = col;
        for (int r = col + 1; r < 3; ++r) if (fabs(M[r][col]) > fabs(M[piv][col])) piv = r;
        if (fabs(M[piv][col]) <= tiny) return 0.0;                      /* singular: G7 */
        if (piv != col) for (int c = 0; c < 4; ++c) { double tmp = M[col][c]; M[col][c] = M[piv][c]; M[piv][c] = tmp; }
        for (int r = col + 1; r < 3; ++r) {
            const double q = M[r][col] / M[col][col];
            for (int c = col; c < 4; ++c) M[r][c] -= q * M[col][c];
        }
    }
    double beta[3];
    for (int r = 2; r >= 0; --r) {
        double v = M[r][3];
        for (int c = r + 1; c < 3; ++c) v -= M[r][c] * beta[c];
        beta[r] = v / M[r][r];
    }
    return beta[0] * rhs[0] + beta[1] * rhs[1] + beta[2] * rhs[2];     /* chi0^2 - chi^2_min */
}

/*
 * Generalised (floating-mean) periodogram, the extension the paper names in section 6.3 (PAPER.md:375,
 * Zechmeister & Kuerster 2009).  Written here as its DEFINITION, not
 * through their closed-form sums: for every frequency, the unweighted linear least-squares fit of
 *     x_j ~ a cos(w t_j) + b sin(w t_j) + c                                (lsp_oracle_gls_fit)
 * and
 *     P = (chi0^2 - chi^2_min) / (2 var),   chi0^2 = sum (x_j - mean)^2,   var = chi0^2 / (Nt - 1)
 * i.e. the same normalisation as eq. (1), which is the special case c = 0: for the 2-function fit
 * the chi^2 reduction IS eq. (1) (pin P1).  0 <= P <= (Nt - 1)/2.  A singular fit (w = 0: the constant and the
 * cosine coincide) returns 0 (reading G7 carried over).
 */
static double lsp_oracle_gls_one(const double* t, const double* X, int64_t Nt, double f, double var)
{
    return lsp_oracle_gls_fit(t, X, NULL, Nt, f) / (2.0 * var);
}

/* Same calling convention as lsp_oracle_periodogram. */
int lsp_oracle_gls(const double* t, const float* x, int64_t Nt,
                   double f_min, double df, const int64_t* ks, int64_t nk,
                   double* P, double* scratch, int nthreads)
{
    double mean, var;
    lsp_oracle_moments(x, Nt, &mean, &var);
    for (int64_t j = 0; j < Nt; ++j) scratch[j] = (double)x[j] - mean;
    int used = 1;
#ifdef _OPENMP
    if (nthreads > 0) omp_set_num_threads(nthreads);
    #pragma omp parallel
    {
        #pragma omp single
        used = omp_get_num_threads();
    }
    #pragma omp parallel for schedule(dynamic, 4)
#endif
    for (int64_t i = 0; i < nk; ++i) {
        int64_t k = ks ? ks[i] : i;
        P[i] = lsp_oracle_gls_one(t, scratch, Nt, f_min + (double)k * df, var);
    }
    return used;
}

/*
 * Weighted generalised periodogram (SURVEY.md 8(f)-1 "optional weights"; the per-sample weights w_j of Zechmeister &
 * Kuerster 2009, the extension the paper names at PAPER.md:375).  Again the DEFINITION, not their closed-form sums:
 * for every frequency, the WEIGHTED linear least-squares fit
 *     minimise  chi^2 = sum_j w_j (x_j - a cos(w t_j) - b sin(w t_j) - c)^2
 * (lsp_oracle_gls_fit), against the weighted constant model
 *     chi0^2 = sum_j w_j (x_j - xbar_w)^2,   xbar_w = sum w_j x_j / sum w_j,
 * and  P = (Nt - 1)/2 * (chi0^2 - chi^2_min) / chi0^2.
 * Reading G14: the paper gives no normalisation for the weighted case; this one is the unweighted
 * P = (chi0^2 - chi^2_min)/(2 var), var = chi0^2/(Nt - 1), written as a chi^2 RATIO, so that w_j = const reproduces
 * lsp_oracle_gls exactly and 0 <= P <= (Nt - 1)/2 whatever the weights.  Only the ratios of the weights matter.
 * Weights must be finite and >= 0 with a positive sum (w_j = 0 removes sample j from the fit but not from Nt).
 */
static double lsp_oracle_gls_w_one(const double* t, const double* X, const double* w, int64_t Nt, double f, double chi0)
{
    return 0.5 * (double)(Nt - 1) * lsp_oracle_gls_fit(t, X, w, Nt, f) / chi0;   /* (X has zero weighted mean) */
}

/* Same calling convention as lsp_oracle_gls plus wts[Nt] fp32 (host) and a second scratch array of Nt doubles. */
int lsp_oracle_gls_weighted(const double* t, const float* x, const float* wts, int64_t Nt,
                            double f_min, double df, const int64_t* ks, int64_t nk,
                            double* P, double* scratch, double* scratch_w, int nthreads)
{
    double sw = 0.0, swx = 0.0;
    for (int64_t j = 0; j < Nt; ++j) { sw += (double)wts[j]; swx += (double)wts[j] * (double)x[j]; }
    const double mean = swx / sw;
    double chi0 = 0.0;
    for (int64_t j = 0; j < Nt; ++j) {
        scratch[j] = (double)x[j] - mean;
        scratch_w[j] = (double)wts[j];
        chi0 += scratch_w[j] * scratch[j] * scratch[j];
    }
    int used = 1;
#ifdef _OPENMP
    if (nthreads > 0) omp_set_num_threads(nthreads);
    #pragma omp parallel
    {
        #pragma omp single
        used = omp_get_num_threads();
    }
    #pragma omp parallel for schedule(dynamic, 4)
#endif
    for (int64_t i = 0; i < nk; ++i) {
        int64_t k = ks ? ks[i] : i;
        P[i] = lsp_oracle_gls_w_one(t, scratch, scratch_w, Nt, f_min + (double)k * df, chi0);
    }
    return used;
}

/* Lowest index among equal maxima (reading G9). */
int64_t lsp_oracle_argmax(const double* P, int64_t n)
{
    int64_t best = 0;
    for (int64_t i = 1; i < n; ++i)
        if (P[i] > P[best]) best = i;
    return best;
}
