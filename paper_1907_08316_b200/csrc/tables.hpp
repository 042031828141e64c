// tables.hpp -- host-side constants of the CUDA library: Gauss-Legendre rule and the
// coefficients of the polynomials A_jl(theta), B_jl(theta).
//
// Deliberately a DIFFERENT route from the CPU oracle (which finds the nodes by Newton
// iteration and integrates A,B by quadrature at run time): here the nodes come from the
// textbook closed forms and A,B are expanded once, in long double, into polynomials in
// theta of degree 2o-1 that the device evaluates by Horner's rule.
//
// Definition restated from the paper ("the L2 projection at the heart of the
// algorithm"; DESIGN.md D:O2): with l_j the Lagrange basis on the o Gauss-Legendre nodes
// xi_j of [0,1] and w_j the weights,
//     A_jl(th) = 1/w_j  int_0^{1-th}  l_j(x) l_l(x+th)   dx
//     B_jl(th) = 1/w_j  int_{1-th}^1  l_j(x) l_l(x+th-1) dx .
// Writing l_j(x) = sum_a c_ja x^a and expanding the shifted factor binomially,
//     A_jl = 1/w_j sum_{a,b} c_ja c_lb sum_{r<=b} C(b,r) th^{b-r} (1-th)^{a+r+1}/(a+r+1)
//     B_jl = 1/w_j sum_{a,b} c_ja c_lb sum_{r<=a} C(a,r) (1-th)^{a-r} th^{r+b+1}/(r+b+1)
// (for B substitute x = eta + 1 - th, eta in [0,th]).
#pragma once
#include <cmath>
#include <vector>

namespace sldg {

constexpr int kMaxOrder = 4;
constexpr int kMaxCoef = 2 * kMaxOrder;   // degree 2o-1 -> 2o coefficients

// o-point Gauss-Legendre rule on [0,1], ascending nodes, sum w = 1.  Closed forms (o<=4).
inline bool gauss_legendre_01(int o, double *xi, double *w) {
    long double r[kMaxOrder], W[kMaxOrder];
    switch (o) {
    case 1: r[0] = 0.0L; W[0] = 2.0L; break;
    case 2: {
        long double a = 1.0L / sqrtl(3.0L);
        r[0] = -a; r[1] = a; W[0] = W[1] = 1.0L;
        break;
    }
    case 3: {
        long double a = sqrtl(3.0L / 5.0L);
        r[0] = -a; r[1] = 0.0L; r[2] = a;
        W[0] = W[2] = 5.0L / 9.0L; W[1] = 8.0L / 9.0L;
        break;
    }
    case 4: {
        long double s = (2.0L / 7.0L) * sqrtl(6.0L / 5.0L);
        long double a = sqrtl(3.0L / 7.0L - s), b = sqrtl(3.0L / 7.0L + s);
        long double wa = (18.0L + sqrtl(30.0L)) / 36.0L, wb = (18.0L - sqrtl(30.0L)) / 36.0L;
        r[0] = -b; r[1] = -a; r[2] = a; r[3] = b;
        W[0] = W[3] = wb; W[1] = W[2] = wa;
        break;
    }
    default: return false;
    }
    for (int j = 0; j < o; ++j) {
        xi[j] = (double)(0.5L * (1.0L + r[j]));
        w[j] = (double)(0.5L * W[j]);
    }
    return true;
}

// Long-double version of the same rule (for the coefficient expansion below).
inline void gauss_legendre_01_ld(int o, long double *xi, long double *w) {
    // recompute in long double: same closed forms
    long double r[kMaxOrder], W[kMaxOrder];
    if (o == 1) { r[0] = 0; W[0] = 2; }
    else if (o == 2) { long double a = 1.0L / sqrtl(3.0L); r[0] = -a; r[1] = a; W[0] = W[1] = 1; }
    else if (o == 3) {
        long double a = sqrtl(0.6L); r[0] = -a; r[1] = 0; r[2] = a;
        W[0] = W[2] = 5.0L / 9.0L; W[1] = 8.0L / 9.0L;
    } else {
        long double s = (2.0L / 7.0L) * sqrtl(1.2L);
        long double a = sqrtl(3.0L / 7.0L - s), b = sqrtl(3.0L / 7.0L + s);
        long double wa = (18.0L + sqrtl(30.0L)) / 36.0L, wb = (18.0L - sqrtl(30.0L)) / 36.0L;
        r[0] = -b; r[1] = -a; r[2] = a; r[3] = b; W[0] = W[3] = wb; W[1] = W[2] = wa;
    }
    for (int j = 0; j < o; ++j) { xi[j] = 0.5L * (1.0L + r[j]); w[j] = 0.5L * W[j]; }
}

// Polynomial helper: p(th) = sum_k c[k] th^k, fixed capacity.
struct PolyLD {
    long double c[kMaxCoef + 2];
    PolyLD() { for (auto &x : c) x = 0.0L; }
};

inline PolyLD poly_mul(const PolyLD &a, const PolyLD &b) {
    PolyLD r;
    for (int i = 0; i < kMaxCoef + 2; ++i)
        for (int k = 0; i + k < kMaxCoef + 2; ++k) r.c[i + k] += a.c[i] * b.c[k];
    return r;
}

// th^e * (1-th)^g
inline PolyLD poly_th_pow_times_one_minus_pow(int e, int g) {
    PolyLD one_minus; one_minus.c[0] = 1.0L; one_minus.c[1] = -1.0L;
    PolyLD r; r.c[0] = 1.0L;
    for (int i = 0; i < g; ++i) r = poly_mul(r, one_minus);
    PolyLD s;
    for (int k = 0; k + e < kMaxCoef + 2; ++k) s.c[k + e] = r.c[k];
    return s;
}

inline long double binom(int n, int k) {
    long double v = 1.0L;
    for (int i = 1; i <= k; ++i) v = v * (long double)(n - k + i) / (long double)i;
    return v;
}

// coef[(((mat*o + j)*o + l)*(2o) + k)*2 + {0,1}] = (hi, lo) double-double pair of the
// coefficient of th^k in A_jl (mat=0) / B_jl (mat=1): hi + lo carries the long-double value,
// so that the device's double-double Horner gives A,B that are "rounded once" (D:O7).
inline std::vector<double> ab_polynomial_coefficients(int o) {
    long double xi[kMaxOrder], w[kMaxOrder];
    gauss_legendre_01_ld(o, xi, w);
    // monomial coefficients of l_j: product of (x - xi_m)/(xi_j - xi_m)
    long double c[kMaxOrder][kMaxOrder];
    for (int j = 0; j < o; ++j) {
        long double p[kMaxOrder + 1] = {1.0L};
        int deg = 0;
        for (int m = 0; m < o; ++m) {
            if (m == j) continue;
            long double d = xi[j] - xi[m];
            long double q[kMaxOrder + 1] = {0};
            for (int k = 0; k <= deg; ++k) {        // p * (x - xi_m) / d
                q[k + 1] += p[k] / d;
                q[k] += -xi[m] * p[k] / d;
            }
            ++deg;
            for (int k = 0; k <= deg; ++k) p[k] = q[k];
        }
        for (int k = 0; k < o; ++k) c[j][k] = p[k];
    }
    const int nc = 2 * o;
    std::vector<double> coef((size_t)2 * o * o * nc * 2, 0.0);
    auto put = [&](size_t idx, long double v) {
        double hi = (double)v;
        coef[idx * 2] = hi;
        coef[idx * 2 + 1] = (double)(v - (long double)hi);
    };
    for (int j = 0; j < o; ++j)
        for (int l = 0; l < o; ++l) {
            PolyLD PA, PB;
            for (int a = 0; a < o; ++a)
                for (int b = 0; b < o; ++b) {
                    long double cc = c[j][a] * c[l][b];
                    for (int r = 0; r <= b; ++r) {
                        PolyLD t = poly_th_pow_times_one_minus_pow(b - r, a + r + 1);
                        long double s = cc * binom(b, r) / (long double)(a + r + 1);
                        for (int k = 0; k < nc; ++k) PA.c[k] += s * t.c[k];
                    }
                    for (int r = 0; r <= a; ++r) {
                        PolyLD t = poly_th_pow_times_one_minus_pow(r + b + 1, a - r);
                        long double s = cc * binom(a, r) / (long double)(r + b + 1);
                        for (int k = 0; k < nc; ++k) PB.c[k] += s * t.c[k];
                    }
                }
            for (int k = 0; k < nc; ++k) {
                put(((size_t)(0 * o + j) * o + l) * nc + k, PA.c[k] / w[j]);
                put(((size_t)(1 * o + j) * o + l) * nc + k, PB.c[k] / w[j]);
            }
            // theta = 0: A = I and B = 0 exactly (int_0^1 l_j l_l = w_j delta_jl because the o-point
            // rule is exact for degree 2o-2), so integer shifts move data bit-exactly (D:R3, P4).
            put(((size_t)(0 * o + j) * o + l) * nc, (j == l) ? 1.0L : 0.0L);
            put(((size_t)(1 * o + j) * o + l) * nc, 0.0L);
        }
    return coef;
}

}  // namespace sldg
