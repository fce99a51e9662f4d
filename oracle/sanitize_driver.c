/*
 * sanitize_driver.c -- TEST INFRASTRUCTURE.  A small main() around oracle_fredec.c for the
 * AddressSanitizer / UndefinedBehaviorSanitizer build that tests/test_oracle_sanitizers.py compiles
 * and runs ("-fsanitize=address,undefined on the oracle").  It calls every
 * entry point of the oracle on small deterministic inputs, including the edge cases (d = 0, the
 * smallest N, a singular trial frequency, fewer peaks than k), and prints the results with 17
 * digits so that the test can compare them with the regular build.
 */
#include <math.h>
#include <stdint.h>
#include <stdio.h>
#include <stdlib.h>

int oracle_scan(const double *t, const double *x, const double *w, int64_t N, const double *base_funcs,
                int32_t d, double f0, double df, int64_t K, double *z_out);
int oracle_chi2_base(const double *t, const double *x, const double *w, int64_t N, const double *base_funcs,
                     int32_t d, double *chi2_base_out);
int oracle_trig_averages(const double *t, const double *x, const double *w, int64_t N, const double *freqs,
                         int64_t M, double *out);
int oracle_topk(const double *z, int64_t K, int32_t k, int64_t *idx_out);

/* a fixed linear congruential sequence in [0, 1): the inputs need no statistical quality */
static uint64_t state = 88172645463325252ULL;
static double next_uniform(void)
{
    state = state * 6364136223846793005ULL + 1442695040888963407ULL;
    return (double)(state >> 11) / 9007199254740992.0;
}

int main(void)
{
    enum { N = 57, D = 4, K = 41, M = 5 };
    double *t = malloc(sizeof(double) * N), *x = malloc(sizeof(double) * N), *w = malloc(sizeof(double) * N);
    double *base = malloc(sizeof(double) * D * N), *z = malloc(sizeof(double) * K);
    double *avg = malloc(sizeof(double) * M * 10);
    int64_t *idx = malloc(sizeof(int64_t) * 8);
    double tt = 0.0;
    for (int i = 0; i < N; ++i) {
        tt += 0.1 + 3.0 * next_uniform();
        t[i] = tt;
        w[i] = 0.25 + next_uniform();
        x[i] = 2.0 * cos(0.7 * tt + 0.3) + next_uniform() - 0.5;
        base[0 * N + i] = 1.0;
        base[1 * N + i] = tt / 100.0;
        base[2 * N + i] = cos(6.283185307179586 * 0.125 * tt);
        base[3 * N + i] = sin(6.283185307179586 * 0.125 * tt);
    }
    int rc = 0;
    double chi2;
    for (int d = 0; d <= D; ++d) {
        rc |= oracle_scan(t, x, w, N, d ? base : NULL, d, 0.0, 0.0125, K, z);
        rc |= oracle_chi2_base(t, x, w, N, d ? base : NULL, d, &chi2);
        printf("scan d=%d chi2=%.17g", d, chi2);
        for (int k = 0; k < K; k += 5) printf(" %.17g", z[k]);
        printf("\n");
        int found = oracle_topk(z, K, 8, idx);
        printf("topk d=%d found=%d", d, found);
        for (int j = 0; j < 8; ++j) printf(" %lld", (long long)idx[j]);
        printf("\n");
    }
    /* smallest N the interface admits (N = d + 3), one grid point */
    double small_base[2 * 5];
    for (int i = 0; i < 5; ++i) {
        small_base[i] = 1.0;
        small_base[5 + i] = t[i];
    }
    rc |= oracle_scan(t, x, w, 2 + 3, small_base, 2, 0.1, 0.1, 1, z);
    printf("small %.17g\n", z[0]);
    /* monotone array: a single peak at the edge, fewer peaks than k */
    for (int k = 0; k < K; ++k) z[k] = (double)k;
    const int edge_found = oracle_topk(z, K, 3, idx);
    printf("edge found=%d idx0=%lld idx1=%lld\n", edge_found, (long long)idx[0], (long long)idx[1]);
    double freqs[M] = {0.0, 0.01, 0.125, 0.77, 3.3};
    rc |= oracle_trig_averages(t, x, w, N, freqs, M, avg);
    for (int j = 0; j < M; ++j) {
        printf("trig %d", j);
        for (int q = 0; q < 10; ++q) printf(" %.17g", avg[j * 10 + q]);
        printf("\n");
    }
    printf("rc=%d\n", rc);
    free(t); free(x); free(w); free(base); free(z); free(avg); free(idx);
    return rc;
}
