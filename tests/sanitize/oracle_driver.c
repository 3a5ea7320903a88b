/* oracle_driver.c -- TEST CODE: calls oracle/sg_oracle.c (both builds, compiled into this program with
 * -fsanitize=address,undefined by tests/test_host_sanitizers.py) on rectangles read from stdin and prints the forces
 * with 17 significant digits, for comparison with the ordinary build of the same source.
 * stdin: n_c n_t slopes(0/1) unit G, then n_c rows "kxl kxr kyd kyu sigma dx dy", then n_t rows "ktx kty". */
#include <stdint.h>
#include <stdio.h>
#include <stdlib.h>

int sg_oracle_force_f80(int64_t, const int64_t *, const int64_t *, const int64_t *, const int64_t *, const double *,
                        const double *, const double *, int64_t, const int64_t *, const int64_t *, double, double,
                        double *, double *, int);
int sg_oracle_force_f64(int64_t, const int64_t *, const int64_t *, const int64_t *, const int64_t *, const double *,
                        const double *, const double *, int64_t, const int64_t *, const int64_t *, double, double,
                        double *, double *, int);

int main(void) {
    long long n_c = 0, n_t = 0;
    int slopes = 0;
    double unit = 0, G = 0;
    if (scanf("%lld %lld %d %lf %lf", &n_c, &n_t, &slopes, &unit, &G) != 5 || n_c < 0 || n_t < 0) return 2;
    int64_t *r = malloc(sizeof(int64_t) * (size_t)(4 * n_c + 2 * n_t + 1));
    double *f = malloc(sizeof(double) * (size_t)(3 * n_c + 4 * n_t + 1));
    if (!r || !f) return 2;
    int64_t *kxl = r, *kxr = r + n_c, *kyd = r + 2 * n_c, *kyu = r + 3 * n_c, *ktx = r + 4 * n_c, *kty = ktx + n_t;
    double *sigma = f, *dx = f + n_c, *dy = f + 2 * n_c, *out = f + 3 * n_c;
    for (long long c = 0; c < n_c; ++c) {
        long long a, b, d, e;
        if (scanf("%lld %lld %lld %lld %lf %lf %lf", &a, &b, &d, &e, &sigma[c], &dx[c], &dy[c]) != 7) return 2;
        kxl[c] = a; kxr[c] = b; kyd[c] = d; kyu[c] = e;
    }
    for (long long t = 0; t < n_t; ++t) {
        long long a, b;
        if (scanf("%lld %lld", &a, &b) != 2) return 2;
        ktx[t] = a; kty[t] = b;
    }
    sg_oracle_force_f80(n_c, kxl, kxr, kyd, kyu, sigma, slopes ? dx : NULL, slopes ? dy : NULL, n_t, ktx, kty, unit, G,
                        out, out + n_t, 2);
    sg_oracle_force_f64(n_c, kxl, kxr, kyd, kyu, sigma, slopes ? dx : NULL, slopes ? dy : NULL, n_t, ktx, kty, unit, G,
                        out + 2 * n_t, out + 3 * n_t, 2);
    for (long long t = 0; t < n_t; ++t)
        printf("%.17g %.17g %.17g %.17g\n", out[t], out[n_t + t], out[2 * n_t + t], out[3 * n_t + t]);
    free(r); free(f);
    return 0;
}
