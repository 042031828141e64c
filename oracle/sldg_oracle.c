/*
 * sldg_oracle.c -- plain CPU oracle (TEST INFRASTRUCTURE, not the product; see
 * sldg_oracle.h for who may call it).  fp64 parts: Gauss-Legendre rule, Lagrange
 * basis, the matrices A(theta), B(theta), the spectral Poisson solve.  The parts
 * that exist for both storage types T (double, float) are in
 * sldg_oracle_real.inc, included twice at the bottom.
 *
 * Written from PAPER.md (P:n) and the readings of SURVEY.md section 8(c)
 * (S:Ox / S:Rx).  No blocking, fusion or reordering beyond what those state;
 * "#pragma omp parallel for" over independent lines / columns is the only
 * concession to run time and does not change any result.
 */
#include "sldg_oracle.h"

#include <float.h>
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

static const double ORACLE_PI = 3.14159265358979323846264338327950288;

/* Guard, not arithmetic: the rule, the A,B quadrature and the rho / mass / l2 / moment sums are "computed in
 * long double and rounded once" (D:O4, D:O7, D:R12), and the pins hold them to 1e-13.  That needs a long double
 * with at least the 64-bit mantissa of x87 extended precision.  Where long double is plain double (MSVC, some
 * ARM ABIs) the sums would silently fall back to the running double sum that the comment above oracle_rho
 * measures as not good enough; refuse to build there instead.  (binary128 long double, e.g. aarch64 Linux,
 * passes: slower, at least as accurate.) */
_Static_assert(LDBL_MANT_DIG >= 64, "the oracle needs long double with >= 64 mantissa bits (x87 extended or wider)");

int oracle_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ---- O1: Gauss-Legendre nodes/weights on [0,1] ------------------------------ */

/* Legendre P_o(r) and P_o'(r) by the three-term recurrence.
 *
 * Precision note (D:O7 / D:R9 "A,B ... rounded once to T"): the nodes, the weights and the
 * matrices A,B are DEFINED as exact real numbers (roots of P_o, exact integrals) that are
 * rounded once.  To make "rounded once" true in practice the rule and the A,B quadrature
 * are carried out in long double (64-bit mantissa on x86) and rounded to double at the
 * end; a plain-double evaluation is off by up to 2 ulp in most entries, which an unstable
 * problem (config 2) amplifies to ~3e-12 between two honest implementations. */
static void legendre_pd(int o, long double r, long double *P, long double *dP) {
    long double p0 = 1.0L, p1 = r;
    if (o == 0) { *P = 1.0L; *dP = 0.0L; return; }
    for (int k = 2; k <= o; ++k) {
        long double p2 = ((2.0L * k - 1.0L) * r * p1 - (k - 1.0L) * p0) / k;
        p0 = p1; p1 = p2;
    }
    *P = p1;
    *dP = o * (r * p1 - p0) / (r * r - 1.0L);
}

static int gauss_legendre_ld(int o, long double *xi, long double *w) {
    if (o < 1 || o > ORACLE_MAX_ORDER || !xi || !w) return 1;
    for (int i = 0; i < o; ++i) {
        /* roots of P_o on [-1,1], descending in i; Newton from the Chebyshev guess */
        long double r = cosl((long double)ORACLE_PI * (i + 0.75L) / (o + 0.5L));
        long double P, dP;
        for (int it = 0; it < 100; ++it) {
            legendre_pd(o, r, &P, &dP);
            long double dr = P / dP;
            r -= dr;
            if (fabsl(dr) < 1e-21L) break;
        }
        legendre_pd(o, r, &P, &dP);
        long double W = 2.0L / ((1.0L - r * r) * dP * dP);
        xi[o - 1 - i] = 0.5L * (1.0L + r);   /* ascending on [0,1] */
        w[o - 1 - i] = 0.5L * W;
    }
    if (o % 2 == 1) xi[o / 2] = 0.5L;        /* the middle root is exactly r = 0 */
    return 0;
}

int oracle_gauss_legendre(int o, double *xi, double *w) {
    long double xl[ORACLE_MAX_ORDER], wl[ORACLE_MAX_ORDER];
    if (!xi || !w || gauss_legendre_ld(o, xl, wl)) return 1;
    for (int j = 0; j < o; ++j) { xi[j] = (double)xl[j]; w[j] = (double)wl[j]; }
    return 0;
}

static long double lagrange_ld(int o, const long double *xi, int j, long double x) {
    long double v = 1.0L;
    for (int m = 0; m < o; ++m)
        if (m != j) v *= (x - xi[m]) / (xi[j] - xi[m]);
    return v;
}

double oracle_lagrange(int o, const double *xi, int j, double x) {
    double v = 1.0;
    for (int m = 0; m < o; ++m)
        if (m != j) v *= (x - xi[m]) / (xi[j] - xi[m]);
    return v;
}

int oracle_node_coords(int n_cells, int o, double lo, double hi, double *c) {
    double xi[ORACLE_MAX_ORDER], w[ORACLE_MAX_ORDER];
    if (n_cells < 1 || !c || oracle_gauss_legendre(o, xi, w)) return 1;
    double h = (hi - lo) / n_cells;
    for (int i = 0; i < n_cells; ++i)
        for (int j = 0; j < o; ++j)
            c[(long)i * o + j] = lo + (i + xi[j]) * h;
    return 0;
}

/* ---- R3: split of the shift ---------------------------------------------------------- */

void oracle_shift_split(double sigma, long *m, double *theta) {
    double delta = -sigma;
    double fl = floor(delta);
    double th = delta - fl;
    /* R3: theta lies in [0,1).  For a tiny negative delta (|delta| < 2^-54: e.g. E = -1e-18 of
     * rounding noise at a node where the field vanishes) the subtraction rounds to exactly 1.0;
     * the translation is continuous across integers (A(1) = 0, B(1) = I equals the next cell with
     * A(0) = I, B(0) = 0), so that case IS the integer shift fl + 1 with theta = 0. */
    if (th >= 1.0) { fl += 1.0; th = 0.0; }
    *m = (long)fl;
    *theta = th;
}

/* ---- O2: A(theta), B(theta) --------------------------------------------- */

int oracle_assemble_AB(int o, double theta_in, double *A, double *B) {
    long double xi[ORACLE_MAX_ORDER], w[ORACLE_MAX_ORDER];
    if (!A || !B || !(theta_in >= 0.0 && theta_in < 1.0)) return 1;
    if (gauss_legendre_ld(o, xi, w)) return 1;
    long double theta = (long double)theta_in;
    long double la = 1.0L - theta;   /* length of [0, 1-theta]  */
    long double lb = theta;          /* length of [1-theta, 1]  */
    for (int j = 0; j < o; ++j) {
        for (int l = 0; l < o; ++l) {
            long double sa = 0.0L, sb = 0.0L;
            for (int q = 0; q < o; ++q) {
                long double xa = la * xi[q];            /* quadrature point in [0, 1-theta] */
                sa += la * w[q] * lagrange_ld(o, xi, j, xa) * lagrange_ld(o, xi, l, xa + theta);
                long double xb = la + lb * xi[q];       /* quadrature point in [1-theta, 1] */
                sb += lb * w[q] * lagrange_ld(o, xi, j, xb) * lagrange_ld(o, xi, l, lb * xi[q]);
            }
            A[j * o + l] = (double)(sa / w[j]);         /* rounded once */
            B[j * o + l] = (double)(sb / w[j]);
        }
    }
    return 0;
}

/* ---- O5 / R6 / R13: spectral Poisson, direct DFT sums --------------------------- */

/* out[.., r, ..] = sum_c (Mre + i Mim)[r][c] * in[.., c, ..] along dimension b of a
 * complex tensor with extents shape[0..nd-1] (index 0 fastest). */
static void cplx_apply_along(const double *in_re, const double *in_im, const long *shape, int nd, int b,
                             const double *Mre, const double *Mim, long rows, double *out_re,
                             double *out_im) {
    long inner = 1, outer = 1, cols = shape[b];
    for (int d = 0; d < b; ++d) inner *= shape[d];
    for (int d = b + 1; d < nd; ++d) outer *= shape[d];
#pragma omp parallel for collapse(2) schedule(static)
    for (long oo = 0; oo < outer; ++oo)
        for (long r = 0; r < rows; ++r)
            for (long ii = 0; ii < inner; ++ii) {
                double sr = 0.0, si = 0.0;
                for (long c = 0; c < cols; ++c) {
                    double xr = in_re[(oo * cols + c) * inner + ii];
                    double xm = in_im[(oo * cols + c) * inner + ii];
                    double mr = Mre[r * cols + c], mi = Mim[r * cols + c];
                    sr += mr * xr - mi * xm;
                    si += mr * xm + mi * xr;
                }
                out_re[(oo * rows + r) * inner + ii] = sr;
                out_im[(oo * rows + r) * inner + ii] = si;
            }
}

int oracle_poisson_E(const double *rho, int dx, const int *cells, int o, const double *lo,
                     const double *hi, double *E) {
    if (!rho || !E || dx < 1 || dx > 3) return 1;
    double xi[ORACLE_MAX_ORDER], w[ORACLE_MAX_ORDER];
    if (oracle_gauss_legendre(o, xi, w)) return 1;

    long Nn[3], K[3], Mmax[3], X = 1, KK = 1;
    double L[3], *c[3] = {0, 0, 0}, *Fre[3], *Fim[3], *Gre[3], *Gim[3];
    for (int a = 0; a < dx; ++a) {
        Nn[a] = (long)cells[a] * o;
        Mmax[a] = (cells[a] - 1) / 2;          /* modes below the cell Nyquist (R6) */
        K[a] = 2 * Mmax[a] + 1;
        L[a] = hi[a] - lo[a];
        X *= Nn[a];
        KK *= K[a];
    }
    /* intermediate tensors are never larger than prod max(N_a, K_a) = X (K_a < N_a) */
    long big = X > KK ? X : KK;
    double *t0r = malloc(sizeof(double) * big), *t0i = malloc(sizeof(double) * big);
    double *t1r = malloc(sizeof(double) * big), *t1i = malloc(sizeof(double) * big);
    double *phr = malloc(sizeof(double) * KK), *phi_ = malloc(sizeof(double) * KK);

    for (int a = 0; a < dx; ++a) {
        c[a] = malloc(sizeof(double) * Nn[a]);
        oracle_node_coords(cells[a], o, lo[a], hi[a], c[a]);
        double h = L[a] / cells[a];
        Fre[a] = malloc(sizeof(double) * K[a] * Nn[a]);
        Fim[a] = malloc(sizeof(double) * K[a] * Nn[a]);
        Gre[a] = malloc(sizeof(double) * K[a] * Nn[a]);
        Gim[a] = malloc(sizeof(double) * K[a] * Nn[a]);
        for (long r = 0; r < K[a]; ++r) {
            double k = 2.0 * ORACLE_PI * (double)(r - Mmax[a]) / L[a];
            for (long p = 0; p < Nn[a]; ++p) {
                double ph = k * c[a][p];
                double wq = w[p % o] * h / L[a];       /* Gauss weight of the node / |Omega_a| */
                Fre[a][r * Nn[a] + p] = wq * cos(ph);  /* forward:  W e^{-i k x} / L            */
                Fim[a][r * Nn[a] + p] = -wq * sin(ph);
                Gre[a][p * K[a] + r] = cos(ph);        /* backward: e^{+i k x}                   */
                Gim[a][p * K[a] + r] = sin(ph);
            }
        }
    }

    /* forward: g_hat(m) = 1/|Omega| sum_x W_x (rho+1)(x) e^{-i k.x}, one dimension at a time */
    long shape[3];
    for (int a = 0; a < dx; ++a) shape[a] = Nn[a];
    for (long x = 0; x < X; ++x) { t0r[x] = rho[x] + 1.0; t0i[x] = 0.0; }
    for (int a = 0; a < dx; ++a) {
        cplx_apply_along(t0r, t0i, shape, dx, a, Fre[a], Fim[a], K[a], t1r, t1i);
        shape[a] = K[a];
        double *s;
        s = t0r; t0r = t1r; t1r = s;
        s = t0i; t0i = t1i; t1i = s;
    }
    /* phi_hat = g_hat / |k|^2, zero mode dropped (R13) */
    for (long q = 0; q < KK; ++q) {
        long rem = q; double k2 = 0.0;
        for (int a = 0; a < dx; ++a) {
            long r = rem % K[a]; rem /= K[a];
            double k = 2.0 * ORACLE_PI * (double)(r - Mmax[a]) / L[a];
            k2 += k * k;
        }
        if (k2 == 0.0) { phr[q] = 0.0; phi_[q] = 0.0; }
        else { phr[q] = t0r[q] / k2; phi_[q] = t0i[q] / k2; }
    }
    /* E_a = Re sum_m (-i k_a) phi_hat(m) e^{+i k.x} */
    for (int a = 0; a < dx; ++a) {
        for (long q = 0; q < KK; ++q) {
            long rem = q, r = 0;
            for (int b = 0; b <= a; ++b) { r = rem % K[b]; rem /= K[b]; }
            double k = 2.0 * ORACLE_PI * (double)(r - Mmax[a]) / L[a];
            /* (-i k)(pr + i pi) = k pi - i k pr */
            t0r[q] = k * phi_[q];
            t0i[q] = -k * phr[q];
        }
        for (int b = 0; b < dx; ++b) shape[b] = K[b];
        for (int b = 0; b < dx; ++b) {
            cplx_apply_along(t0r, t0i, shape, dx, b, Gre[b], Gim[b], Nn[b], t1r, t1i);
            shape[b] = Nn[b];
            double *s;
            s = t0r; t0r = t1r; t1r = s;
            s = t0i; t0i = t1i; t1i = s;
        }
        for (long x = 0; x < X; ++x) E[(long)a * X + x] = t0r[x];
    }

    for (int a = 0; a < dx; ++a) { free(c[a]); free(Fre[a]); free(Fim[a]); free(Gre[a]); free(Gim[a]); }
    free(t0r); free(t0i); free(t1r); free(t1i); free(phr); free(phi_);
    return 0;
}

/* ---- the parts that exist per storage type T ------------------------------------------ */

#define REAL double
#define SUF(name) name##_f64
#define REAL_FMA(a, b, c) fma((a), (b), (c))
#include "sldg_oracle_real.inc"
#undef REAL
#undef SUF
#undef REAL_FMA

#define REAL float
#define SUF(name) name##_f32
#define REAL_FMA(a, b, c) fmaf((a), (b), (c))
#include "sldg_oracle_real.inc"
#undef REAL
#undef SUF
#undef REAL_FMA
