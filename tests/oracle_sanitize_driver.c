/* Test infrastructure (SURVEY 4 tier T4, CPU part): drives every entry point of oracle/colatus_oracle.c on small
 * heap-allocated inputs of exact size, so that AddressSanitizer / UBSan (tests/test_oracle_sanitizers.py builds
 * this file together with the oracle under -fsanitize=address,undefined) see any out-of-bounds access, use of
 * uninitialised heap padding or undefined arithmetic.  Prints "sanitize-ok <checksum>" on success. */
#include <math.h>
#include <stdint.h>
#include <stdio.h>
#include <stdlib.h>

void oracle_forces(const double *, const double *, int64_t, double, double, const int64_t *, int64_t, double *, double *);
void oracle_step(double *, double *, const double *, int64_t, double, double, double, double, double, double *);
void oracle_step_coeffs(double *, double *, const double *, int64_t, double, double, double, double, double, double,
                        double *);
void oracle_add_external(const double *, const int64_t *, int64_t, double, double, const double *, double, double,
                         const double *, double *);
void oracle_step_coeffs_ext(double *, double *, const double *, int64_t, double, double, double, double, double, double,
                            double, const double *, double, const double *, double *);
double oracle_hubble(double, double, double, double, double, double);
double oracle_a_advance(double, double, double, double, double, double, double, int);
double oracle_time_of_a(double, double, double, double, double, double, int64_t);
double oracle_int_dt_over_a_pow(double, double, double, double, double, double, double, double, int);
void oracle_diagnostics(const double *, const double *, const double *, int64_t, double, double, double, int, double *);
void oracle_splat(const float *, int64_t, int, const float *, int, int, uint32_t *);
void oracle_trace_spectrum(const float *, int64_t, int64_t, double *);

static uint64_t lcg = 88172645463325252ULL;
static double urand(void) {
    lcg = lcg * 6364136223846793005ULL + 1442695040888963407ULL;
    return (double)(lcg >> 11) / 9007199254740992.0;
}

int main(void) {
    const int64_t sizes[4] = {1, 2, 33, 257};
    double sum = 0.0;
    for (int s = 0; s < 4; ++s) {
        const int64_t n = sizes[s];
        double *x = malloc(sizeof(double) * 3 * n), *v = malloc(sizeof(double) * 3 * n), *m = malloc(sizeof(double) * n);
        double *acc = malloc(sizeof(double) * 3 * n), *phi = malloc(sizeof(double) * n), *work = malloc(sizeof(double) * 3 * n);
        int64_t *tg = malloc(sizeof(int64_t) * n);
        float *pmf = malloc(sizeof(float) * 4 * n);
        for (int64_t i = 0; i < n; ++i) {
            for (int c = 0; c < 3; ++c) {
                x[3 * i + c] = urand();
                v[3 * i + c] = 0.1 * (urand() - 0.5);
                pmf[4 * i + c] = (float)x[3 * i + c];
            }
            m[i] = (0.5 + urand()) / n;
            pmf[4 * i + 3] = (float)m[i];
            tg[i] = n - 1 - i;                                    /* a permuted target list */
        }
        oracle_forces(x, m, n, 1e-4, 1.0, NULL, n, acc, phi);     /* all targets, with potential */
        oracle_forces(x, m, n, 1e-4, 1.0, tg, n, acc, NULL);      /* explicit list, no potential */
        oracle_forces(x, m, n, 1e-4, 1.0, tg, 1, acc, phi);       /* a single target */
        const double xpsi[3] = {0.3, 0.4, 0.5}, cen[3] = {0.5, 0.5, 0.5};
        oracle_add_external(x, tg, n, 1e-4, 0.2, xpsi, 1.0, 1.0, cen, acc);
        oracle_add_external(x, NULL, n, 1e-4, 0.0, xpsi, 1.0, 0.5, cen, acc);
        oracle_step(x, v, m, n, 1e-4, 1.0, 1e-3, 0.5, 0.7, work);
        oracle_step_coeffs(x, v, m, n, 1e-4, 1.0, 5e-4, 0.99, 1e-3, 5e-4, work);
        oracle_step_coeffs_ext(x, v, m, n, 1e-4, 1.0, 5e-4, 0.99, 1e-3, 5e-4, 0.2, xpsi, 1.0, cen, work);
        double d[16];
        oracle_diagnostics(x, v, m, n, 1e-4, 1.0, 0.5, 1, d);
        oracle_diagnostics(x, v, m, n, 1e-4, 1.0, 0.5, 0, d);
        for (int axis = 0; axis < 3; ++axis) {
            const int W = 7, H = 5;
            const float win[6] = {0.f, 1.f, 0.f, 1.f, 0.25f, 0.75f};
            uint32_t *img = malloc(sizeof(uint32_t) * W * H);
            oracle_splat(pmf, n, axis, win, W, H, img);
            for (int p = 0; p < W * H; ++p) sum += img[p];
            free(img);
        }
        for (int64_t i = 0; i < 3 * n; ++i) sum += x[i] + v[i] + acc[i];
        sum += d[0] + d[7];
        free(x); free(v); free(m); free(acc); free(phi); free(work); free(tg); free(pmf);
    }
    /* tracer periodogram: odd and even lengths, exact-size buffers */
    const int64_t lens[3] = {2, 9, 16};
    for (int s = 0; s < 3; ++s) {
        const int64_t S = lens[s], k = 3;
        float *ser = malloc(sizeof(float) * 4 * S * k);
        double *out = malloc(sizeof(double) * k * (S / 2 + 1));
        for (int64_t i = 0; i < 4 * S * k; ++i) ser[i] = (float)(urand() - 0.5);
        oracle_trace_spectrum(ser, S, k, out);
        for (int64_t i = 0; i < k * (S / 2 + 1); ++i) sum += out[i];
        free(ser); free(out);
    }
    /* eq. (2) helpers */
    sum += oracle_hubble(70.0, 1e-4, 0.3, 0.0, 0.7, 0.5);
    sum += oracle_a_advance(70.0, 1e-4, 0.3, 0.0, 0.7, 0.02, 1e-4, 64);
    sum += oracle_time_of_a(70.0, 1e-4, 0.3, 0.0, 0.7, 1.0, 20000);
    sum += oracle_int_dt_over_a_pow(70.0, 0.0, 0.3, 0.0, 0.7, 0.02, 1e-4, 2.0, 64);
    if (!isfinite(sum)) { printf("non-finite checksum\n"); return 1; }
    printf("sanitize-ok %.6g\n", sum);
    return 0;
}
