/* ASan/UBSan driver for the CPU oracle (SURVEY section 5 "race detection / sanitizers"): every
 * oracle entry point on small RAGGED problems (odd cell counts, every order, 1..3 + 1..3 dimensions,
 * huge and negative shifts, both storage types).  Built by tests/test_oracle_sanitizers.py with
 *   gcc -fsanitize=address,undefined -fno-sanitize-recover=all
 * and run; any out-of-bounds access, use-after-free, leak, signed overflow or misaligned access aborts
 * with a non-zero exit status.  Test infrastructure, like the oracle itself. */
#include <math.h>
#include <stdio.h>
#include <stdlib.h>

#include "../../oracle/sldg_oracle.h"

static double urand(unsigned long long *s) {
    *s = *s * 6364136223846793005ULL + 1442695040888963407ULL;
    return (double)(*s >> 11) * (1.0 / 9007199254740992.0);
}

#define CHECK(call) do { int rc_ = (call); if (rc_) { fprintf(stderr, "%s -> %d\n", #call, rc_); return 2; } } while (0)

static int run_case(int dx, int dv, const int *cells, int o, unsigned long long seed) {
    int D = dx + dv;
    double lo[6], hi[6];
    long N[6], X = 1, total = 1;
    for (int d = 0; d < D; ++d) {
        lo[d] = d < dx ? 0.25 * d : -4.0 - 0.5 * d;
        hi[d] = d < dx ? 2.0 + d : 4.5 + 0.25 * d;
        N[d] = (long)cells[d] * o;
        total *= N[d];
        if (d < dx) X *= N[d];
    }
    double *f = malloc(sizeof(double) * total);
    float *g = malloc(sizeof(float) * total);
    for (long i = 0; i < total; ++i) { f[i] = urand(&seed); g[i] = (float)f[i]; }
    double *rho = malloc(sizeof(double) * X), *E = malloc(sizeof(double) * X * dx);

    /* raw sweeps along every dimension with shifts of either sign, some huge, some integer */
    for (int k = 0; k < D; ++k) {
        int dep[3], ndep;
        long count = 1;
        if (k < dx) { dep[0] = dx + k; ndep = 1; count = N[dx + k]; }
        else { ndep = dx; for (int a = 0; a < dx; ++a) { dep[a] = a; count *= N[a]; } }
        double *sigma = malloc(sizeof(double) * count);
        for (long q = 0; q < count; ++q) sigma[q] = -3.5 + 7.0 * urand(&seed);
        sigma[0] = 1e9 + 0.5; sigma[count - 1] = -2.0; if (count > 2) sigma[1] = -1e-300;
        CHECK(oracle_translate_f64(f, D, N, o, k, sigma, ndep, dep));
        CHECK(oracle_translate_f32(g, D, N, o, k, sigma, ndep, dep));
        free(sigma);
    }
    CHECK(oracle_rho_f64(f, dx, dv, cells, o, lo, hi, rho));
    CHECK(oracle_rho_f32(g, dx, dv, cells, o, lo, hi, rho));
    CHECK(oracle_poisson_E(rho, dx, cells, o, lo, hi, E));
    for (int k = 0; k < D; ++k) {
        if (k >= dx && k - dx >= dx) continue;             /* v_a without a field component */
        CHECK(oracle_advect_f64(f, dx, dv, cells, o, lo, hi, k, 0.37, E));
        CHECK(oracle_advect_f32(g, dx, dv, cells, o, lo, hi, k, 0.37, E));
    }
    CHECK(oracle_step_f64(f, dx, dv, cells, o, lo, hi, 0.1));
    CHECK(oracle_step_f32(g, dx, dv, cells, o, lo, hi, 0.1));
    double mass, l2, ee, P[3], K;
    CHECK(oracle_diagnostics_f64(f, dx, dv, cells, o, lo, hi, &mass, &l2, &ee));
    CHECK(oracle_diagnostics_f32(g, dx, dv, cells, o, lo, hi, &mass, &l2, &ee));
    CHECK(oracle_moments_f64(f, dx, dv, cells, o, lo, hi, P, &K));
    CHECK(oracle_moments_f32(g, dx, dv, cells, o, lo, hi, P, &K));
    if (!(mass > 0.0) || !(l2 > 0.0) || !(ee >= 0.0) || !isfinite(K)) { fprintf(stderr, "bad invariants\n"); return 3; }
    free(f); free(g); free(rho); free(E);
    return 0;
}

int main(void) {
    /* the small building blocks */
    for (int o = 1; o <= 6; ++o) {
        double xi[8], w[8], A[64], B[64], c[64];
        CHECK(oracle_gauss_legendre(o, xi, w));
        for (int t = 0; t < 5; ++t) CHECK(oracle_assemble_AB(o, t == 4 ? 1.0 - 0x1p-53 : 0.25 * t, A, B));
        CHECK(oracle_node_coords(7, o, -1.0, 2.5, c));
        (void)oracle_lagrange(o, xi, o - 1, 0.3);
        long m; double th;
        oracle_shift_split(-1e-300, &m, &th);
        oracle_shift_split(123456789.25, &m, &th);
        if (oracle_assemble_AB(o, 1.0, A, B) == 0) { fprintf(stderr, "theta = 1 must be rejected\n"); return 4; }
    }
    const int c11[2] = {7, 5}, c12[3] = {5, 3, 4}, c22[4] = {5, 3, 4, 3}, c13[4] = {4, 3, 2, 3};
    const int c23[5] = {3, 4, 3, 2, 3}, c33[6] = {3, 2, 3, 2, 3, 2};
    int rc = 0;
    for (int o = 1; o <= 6 && !rc; ++o) rc = run_case(1, 1, c11, o, 11 + o);
    for (int o = 1; o <= 4 && !rc; ++o) rc = run_case(2, 2, c22, o, 22 + o);
    if (!rc) rc = run_case(1, 2, c12, 3, 12);
    if (!rc) rc = run_case(1, 3, c13, 2, 13);
    if (!rc) rc = run_case(2, 3, c23, 2, 23);
    if (!rc) rc = run_case(3, 3, c33, 2, 33);
    if (!rc) rc = run_case(3, 3, c33, 1, 34);
    if (rc) return rc;
    puts("oracle sanitizer run: ok");
    return 0;
}
