/*
 * oracle_fredec.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, obviously-correct CPU implementation of the single-frequency residual
 * periodogram of FREDEC (Baluev 2013, arXiv:1309.0100), written from the paper.  Only
 * tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
 * may call it.  It shares no code, header, table or helper with the CUDA path under
 * paper_1309_0100_b200/csrc/ and neither includes the other.
 *
 * What it computes, for every grid frequency f_k = f0 + k*df  (k = 0..K-1):
 *
 *   z(f) = min_theta chi2_base(theta)  -  min_{theta,a,b} chi2_alt(theta,a,b; f)
 *
 *   chi2 = <(x - mu)^2>,  <phi> = sum_i w_i phi(t_i)      PAPER.md:62 (eq. 3), :67 (eq. 4)
 *   mu_base = sum_j theta_j phi_j(t)                      PAPER.md:49-56 (eqs. 1, 2), :51
 *   mu_alt  = mu_base + a cos(2 pi f t) + b sin(2 pi f t) PAPER.md:106 (eq. 10, n = 1):
 *             base functions fixed, all d+2 linear coefficients fitted exactly (eq. 5, :72)
 *
 * How (section 3): build g = <x Phi> and Q = <Phi Phi^T> with
 * Phi = (phi_0..phi_{d-1}, cos wt, sin wt), w = 2 pi f (eqs. 15, 16 at PAPER.md:165-171),
 * Cholesky Q = L L^T, forward substitution a = L^{-1} g, and D - l = |a|^2
 * (reading G2 of DESIGN.md: the printed factors 1/2 are inconsistent with
 * eqs. 15-16, plain least squares is meant).  Because the base block is the leading
 * ("low-top") submatrix of Q, its Cholesky factor is the leading block of L:
 * a_0..a_{d-1} are the base model's share of D - l and
 *
 *   z(f) = a_d^2 + a_{d+1}^2,        chi2_base = D - sum_{j<d} a_j^2,   D = <x^2>.
 *
 * sin/cos are evaluated PER PAIR with libm on an exactly range-reduced phase
 * (frac(f*t) through an FMA split), sums run in index order, nothing is blocked, fused
 * or reordered.  The d x d base block of Q and the base part of g do not depend on f and
 * are summed once (same numbers as re-summing them for every k).
 *
 * Readings the paper leaves open: grid frequency = fl(fma(k,df,f0))
 * (S1); singular trial system rule (S6); peak definition and order (S7).  PARITY
 * UNPINNED BY THE PAPER for those three: they are this build's decisions.
 *
 * Build variants (oracle/build.py): ORACLE_REAL=double (the oracle), ORACLE_REAL=long
 * double with ORACLE_SUFFIX=_ld (80-bit, measures the oracle's own rounding error);
 * -fopenmp parallelises ONLY the k loop (each frequency is still summed sequentially,
 * hence bit-identical to the serial run).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#ifndef ORACLE_REAL
#define ORACLE_REAL double
#define ORACLE_IS_DOUBLE 1
#endif
#ifndef ORACLE_SUFFIX
#define ORACLE_SUFFIX
#endif

typedef ORACLE_REAL real;

#ifdef ORACLE_IS_DOUBLE
#define R_FMA fma
#define R_RINT rint
#define R_COS cos
#define R_SIN sin
#define R_SQRT sqrt
#define R_TWO_PI 6.283185307179586476925286766559
#else
#define R_FMA fmal
#define R_RINT rintl
#define R_COS cosl
#define R_SIN sinl
#define R_SQRT sqrtl
#define R_TWO_PI 6.283185307179586476925286766559005768L
#endif

#define CAT2(a, b) a##b
#define CAT(a, b) CAT2(a, b)
#define FN(name) CAT(name, ORACLE_SUFFIX)

#define ORACLE_OK 0
#define ORACLE_EINVAL (-1)
#define ORACLE_ESINGULAR (-3)

/* S6: a trial pivot is dropped when pivot^2 <= TAU * (its un-projected diagonal). */
#define ORACLE_TAU_TRIAL 1e-10
/* base functions count as linearly dependent when pivot^2 <= TAU * diagonal */
#define ORACLE_TAU_BASE 1e-12

/* cos and sin of 2 pi f t with the phase reduced exactly: f*t = hi + lo exactly (FMA),
 * hi - rint(hi) is exact, so the reduced phase carries only the final rounding. */
static void trial_pair(real f, real t, real *c, real *s)
{
    real hi = f * t;
    real lo = R_FMA(f, t, -hi);
    real ph = (hi - R_RINT(hi)) + lo; /* in turns, |ph| <= 1/2 */
    *c = R_COS((real)R_TWO_PI * ph);
    *s = R_SIN((real)R_TWO_PI * ph);
}

/* Lower Cholesky Q = L L^T (in place, row-major n x n, lower triangle) and a = L^{-1} g
 * (in place in g).  Columns >= first_trial are the trial cos/sin columns
 * and obey rule S6; a dependent base column returns ORACLE_ESINGULAR. */
static int cholesky_forward(real *Q, real *g, int n, int first_trial)
{
    for (int j = 0; j < n; ++j) {
        real diag = Q[j * n + j];
        real piv2 = diag;
        for (int m = 0; m < j; ++m) piv2 -= Q[j * n + m] * Q[j * n + m];
        int drop = 0;
        if (j >= first_trial) {
            if (!(piv2 > (real)ORACLE_TAU_TRIAL * diag)) drop = 1;
        } else {
            if (!(piv2 > (real)ORACLE_TAU_BASE * diag)) return ORACLE_ESINGULAR;
        }
        if (drop) { /* column j leaves the model: zero column, zero coefficient */
            Q[j * n + j] = 0;
            for (int r = j + 1; r < n; ++r) Q[r * n + j] = 0;
            g[j] = 0;
            continue;
        }
        real Ljj = R_SQRT(piv2);
        Q[j * n + j] = Ljj;
        for (int r = j + 1; r < n; ++r) {
            real v = Q[r * n + j];
            for (int m = 0; m < j; ++m) v -= Q[r * n + m] * Q[j * n + m];
            Q[r * n + j] = v / Ljj;
        }
        real a = g[j];
        for (int m = 0; m < j; ++m) a -= Q[j * n + m] * g[m];
        g[j] = a / Ljj;
    }
    return ORACLE_OK;
}

static int check_args(const double *t, const double *x, const double *w, int64_t N,
                      const double *base_funcs, int32_t d)
{
    if (!t || !x || !w || d < 0 || (d > 0 && !base_funcs) || N < (int64_t)d + 3) return ORACLE_EINVAL;
    return ORACLE_OK;
}

/* base block of Q (d x d into the n x n array) and base part of g; D = <x^2> */
static void base_block(const double *x, const double *w, int64_t N, const double *base_funcs,
                       int d, int n, real *Q, real *g, real *D)
{
    for (int a = 0; a < n * n; ++a) Q[a] = 0;
    for (int a = 0; a < n; ++a) g[a] = 0;
    real DD = 0;
    for (int64_t i = 0; i < N; ++i) {
        real wi = w[i], xi = x[i];
        DD += wi * xi * xi;
        for (int a = 0; a < d; ++a) {
            real pa = base_funcs[(int64_t)a * N + i];
            g[a] += wi * xi * pa;
            for (int b = 0; b <= a; ++b) Q[a * n + b] += wi * pa * (real)base_funcs[(int64_t)b * N + i];
        }
    }
    *D = DD;
}

/* chi2_base = D - sum_{j<d} a_j^2 : the minimum of chi2 over the base model alone. */
int FN(oracle_chi2_base)(const double *t, const double *x, const double *w, int64_t N,
                         const double *base_funcs, int32_t d, double *chi2_base_out)
{
    int rc = check_args(t, x, w, N, base_funcs, d);
    if (rc || !chi2_base_out) return ORACLE_EINVAL;
    int n = d > 0 ? d : 1;
    real *Q = (real *)malloc(sizeof(real) * n * n), *g = (real *)malloc(sizeof(real) * n), D;
    base_block(x, w, N, base_funcs, d, n, Q, g, &D);
    rc = d > 0 ? cholesky_forward(Q, g, d, d) : ORACLE_OK;
    real l = D;
    for (int j = 0; j < d; ++j) l -= g[j] * g[j];
    *chi2_base_out = (double)l;
    free(Q); free(g);
    return rc;
}

int FN(oracle_scan)(const double *t, const double *x, const double *w, int64_t N,
                    const double *base_funcs, int32_t d, double f0, double df, int64_t K,
                    double *z_out)
{
    int rc = check_args(t, x, w, N, base_funcs, d);
    if (rc || !z_out || K < 1 || !(df > 0) || !(f0 >= 0)) return ORACLE_EINVAL;
    const int n = d + 2;
    real *Qb = (real *)malloc(sizeof(real) * n * n), *gb = (real *)malloc(sizeof(real) * n), D;
    base_block(x, w, N, base_funcs, d, n, Qb, gb, &D);
    int status = ORACLE_OK;

#ifdef _OPENMP
#pragma omp parallel
#endif
    {
        real *Q = (real *)malloc(sizeof(real) * n * n), *g = (real *)malloc(sizeof(real) * n);
#ifdef _OPENMP
#pragma omp for schedule(static)
#endif
        for (int64_t k = 0; k < K; ++k) {
            const real f = (real)fma((double)k, df, f0); /* S1: the grid frequency is a double */
            memcpy(Q, Qb, sizeof(real) * n * n);
            memcpy(g, gb, sizeof(real) * n);
            real *Qc = Q + d * n, *Qs = Q + (d + 1) * n; /* rows of cos and sin */
            for (int64_t i = 0; i < N; ++i) {
                real c, s;
                trial_pair(f, (real)t[i], &c, &s);
                real wi = w[i], xi = x[i];
                for (int b = 0; b < d; ++b) {                 /* <phi_b cos>, <phi_b sin> */
                    real pb = base_funcs[(int64_t)b * N + i];
                    Qc[b] += wi * pb * c;
                    Qs[b] += wi * pb * s;
                }
                Qc[d] += wi * c * c;                           /* <cos^2>      eq. 16 */
                Qs[d] += wi * s * c;                           /* <sin cos>           */
                Qs[d + 1] += wi * s * s;                       /* <sin^2>             */
                g[d] += wi * xi * c;                           /* <x cos>      eq. 15 */
                g[d + 1] += wi * xi * s;                       /* <x sin>             */
            }
            int r = cholesky_forward(Q, g, n, d);
            if (r) {
#ifdef _OPENMP
#pragma omp atomic write
#endif
                status = r;
                z_out[k] = 0.0;
            } else {
                z_out[k] = (double)(g[d] * g[d] + g[d + 1] * g[d + 1]);
            }
        }
        free(Q); free(g);
    }
    free(Qb); free(gb);
    return status;
}

/* Trigonometric averages of PAPER.md:242-262 (section 5) at an arbitrary list of M frequencies
 * (omega_j = 2 pi f_j), per pair with libm on the exactly reduced phase, summed in index order.
 * out [M][10], in the paper's order: system (19)
 *   0 <cos wt>   1 <sin wt>   2 <t cos wt>   3 <t sin wt>
 *   4 <x cos wt> 5 <x sin wt> 6 <x t cos wt> 7 <x t sin wt>
 * and the two further averages of system (20) (its first four are 0..3 above)
 *   8 <t^2 cos wt>  9 <t^2 sin wt>.
 * <phi> = sum_i w_i phi(t_i); t is used as given (the paper sets <t> = 0). */
int FN(oracle_trig_averages)(const double *t, const double *x, const double *w, int64_t N,
                             const double *freqs, int64_t M, double *out)
{
    if (!t || !x || !w || !freqs || !out || N < 1 || M < 1) return ORACLE_EINVAL;
    for (int64_t j = 0; j < M; ++j) {
        real a[10] = {0, 0, 0, 0, 0, 0, 0, 0, 0, 0};
        for (int64_t i = 0; i < N; ++i) {
            real c, s;
            trial_pair((real)freqs[j], (real)t[i], &c, &s);
            const real wi = w[i], ti = t[i], xi = x[i];
            a[0] += wi * c;            a[1] += wi * s;
            a[2] += wi * ti * c;       a[3] += wi * ti * s;
            a[4] += wi * xi * c;       a[5] += wi * xi * s;
            a[6] += wi * xi * ti * c;  a[7] += wi * xi * ti * s;
            a[8] += wi * ti * ti * c;  a[9] += wi * ti * ti * s;
        }
        for (int q = 0; q < 10; ++q) out[j * 10 + q] = (double)a[q];
    }
    return ORACLE_OK;
}

#ifdef ORACLE_IS_DOUBLE
/* Peaks (S7): k is a peak iff z[k] > z[k-1] and z[k] >= z[k+1], neighbours outside the
 * grid count as -infinity, NaN counts as -infinity.  Ranked by z descending, then index
 * ascending; the first k go to idx_out, unused slots are -1.  Returns the number found. */
typedef struct { double z; int64_t idx; } peak_t;

static double peak_val(const double *z, int64_t K, int64_t i)
{
    if (i < 0 || i >= K) return -INFINITY;
    return isnan(z[i]) ? -INFINITY : z[i];
}

static int peak_cmp(const void *pa, const void *pb)
{
    const peak_t *a = (const peak_t *)pa, *b = (const peak_t *)pb;
    if (a->z > b->z) return -1;
    if (a->z < b->z) return 1;
    return (a->idx > b->idx) - (a->idx < b->idx);
}

int oracle_topk(const double *z, int64_t K, int32_t k, int64_t *idx_out)
{
    if (!z || !idx_out || K < 1 || k < 1 || k > K) return ORACLE_EINVAL;
    peak_t *peaks = (peak_t *)malloc(sizeof(peak_t) * (size_t)K);
    int64_t n = 0;
    for (int64_t i = 0; i < K; ++i) {
        double v = peak_val(z, K, i);
        if (v > peak_val(z, K, i - 1) && v >= peak_val(z, K, i + 1)) {
            peaks[n].z = v; peaks[n].idx = i; ++n;
        }
    }
    qsort(peaks, (size_t)n, sizeof(peak_t), peak_cmp);
    int found = n < k ? (int)n : k;
    for (int j = 0; j < k; ++j) idx_out[j] = j < found ? peaks[j].idx : -1;
    free(peaks);
    return found;
}

/* threads a parallel loop can use on this machine: the processors available to the process, capped by
 * OMP_NUM_THREADS at start-up -- NOT the value of the last oracle_set_threads call */
int oracle_num_threads(void)
{
#ifdef _OPENMP
    static int at_start = 0;
    if (at_start == 0) at_start = omp_get_max_threads();
    return at_start < omp_get_num_procs() ? at_start : omp_get_num_procs();
#else
    return 1;
#endif
}

void oracle_set_threads(int n)
{
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}
#endif /* ORACLE_IS_DOUBLE */
