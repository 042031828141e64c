// tables.hpp -- host-side constants of the CUDA library: Gauss-Legendre rule and the
// coefficients of the polynomials A_jl(theta), B_jl(theta).
//
// Deliberately a DIFFERENT route from the CPU oracle (which finds the nodes by Newton
// iteration and integrates A,B by quadrature at run time): here the nodes come from closed
// forms (roots of P_o by radicals / the trigonometric solution of a cubic) and A,B are
// expanded once, in binary128 (__float128, host only), into polynomials in theta of degree
// 2o-1 that the device evaluates by double-double Horner.
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
//
// Why binary128: the monomial coefficients grow to ~1e5 at o = 6 and cancel; "A,B rounded
// once" (D:O7) needs them good to well below one ulp of the O(1) result.
#pragma once
#include <cmath>
#include <vector>

namespace sldg {

typedef __float128 q128;

constexpr int kMaxOrder = 6;
constexpr int kMaxCoef = 2 * kMaxOrder;   // degree 2o-1 -> 2o coefficients

inline q128 q_sqrt(q128 a) {
    if (a <= 0) return 0;
    q128 x = (q128)sqrtl((long double)a);
    for (int i = 0; i < 3; ++i) x = (x + a / x) / 2;     // Newton from a 64-bit start: > 113 bits
    return x;
}

// cos(acos(c)/3 + shift) in binary128: long-double start, then Newton on the triple-angle
// identity 4 y^3 - 3 y = c (y = cos(phi/3 + 2 pi k/3) are its three roots).
inline q128 q_cos_third(q128 c, int k) {
    const long double PI = 3.14159265358979323846264338327950288L;
    long double phi = acosl((long double)c);
    q128 y = (q128)cosl((phi + 2.0L * PI * k) / 3.0L);
    for (int i = 0; i < 4; ++i) y -= (4 * y * y * y - 3 * y - c) / (12 * y * y - 3);
    return y;
}

// Legendre P_o and P_o' at r (three-term recurrence), for the weights 2 / ((1-r^2) P_o'(r)^2)
inline void q_legendre(int o, q128 r, q128 *P, q128 *dP) {
    q128 p0 = 1, p1 = r;
    for (int k = 2; k <= o; ++k) {
        q128 p2 = ((2 * k - 1) * r * p1 - (k - 1) * p0) / k;
        p0 = p1; p1 = p2;
    }
    *P = p1;
    *dP = o * (r * p1 - p0) / (r * r - 1);
}

// o-point Gauss-Legendre rule on [0,1] in binary128, ascending nodes, sum w = 1.
// Roots of P_o on [-1,1] in closed form:
//   o=1: 0            o=2: +-1/sqrt3            o=3: 0, +-sqrt(3/5)
//   o=4: +-sqrt(3/7 -+ (2/7) sqrt(6/5))         o=5: 0, +-(1/3) sqrt(5 -+ 2 sqrt(10/7))
//   o=6: x^2 = t, 231 t^3 - 315 t^2 + 105 t - 5 = 0 (three real roots, trigonometric form)
inline bool gauss_legendre_01_q(int o, q128 *xi, q128 *w) {
    q128 pos[3];            // the positive roots, ascending
    int npos = o / 2;
    switch (o) {
    case 1: break;
    case 2: pos[0] = 1 / q_sqrt(3); break;
    case 3: pos[0] = q_sqrt((q128)3 / 5); break;
    case 4: {
        q128 s = ((q128)2 / 7) * q_sqrt((q128)6 / 5);
        pos[0] = q_sqrt((q128)3 / 7 - s); pos[1] = q_sqrt((q128)3 / 7 + s);
        break;
    }
    case 5: {
        q128 s = 2 * q_sqrt((q128)10 / 7);
        pos[0] = q_sqrt(5 - s) / 3; pos[1] = q_sqrt(5 + s) / 3;
        break;
    }
    case 6: {
        // t^3 + a2 t^2 + a1 t + a0 = 0 with a2 = -315/231, a1 = 105/231, a0 = -5/231;
        // t = s - a2/3 gives s^3 + p s + q = 0, s_k = 2 sqrt(-p/3) cos(acos(3q/(2p) sqrt(-3/p))/3 - 2 pi k/3)
        q128 a2 = -(q128)315 / 231, a1 = (q128)105 / 231, a0 = -(q128)5 / 231;
        q128 p = a1 - a2 * a2 / 3, q = 2 * a2 * a2 * a2 / 27 - a2 * a1 / 3 + a0;
        q128 amp = 2 * q_sqrt(-p / 3), arg = (3 * q) / (2 * p) * q_sqrt(-3 / p);
        q128 t[3];
        for (int k = 0; k < 3; ++k) t[k] = amp * q_cos_third(arg, k) - a2 / 3;
        for (int i = 0; i < 3; ++i)                       // sort ascending
            for (int j = i + 1; j < 3; ++j)
                if (t[j] < t[i]) { q128 x = t[i]; t[i] = t[j]; t[j] = x; }
        for (int k = 0; k < 3; ++k) pos[k] = q_sqrt(t[k]);
        break;
    }
    default: return false;
    }
    q128 r[kMaxOrder];
    for (int k = 0; k < npos; ++k) { r[npos - 1 - k] = -pos[k]; r[o - npos + k] = pos[k]; }
    if (o % 2) r[npos] = 0;
    for (int j = 0; j < o; ++j) {
        q128 P, dP;
        q_legendre(o, r[j], &P, &dP);
        xi[j] = (1 + r[j]) / 2;
        w[j] = 1 / ((1 - r[j] * r[j]) * dP * dP);         // (2 / ...) / 2
    }
    return true;
}

inline bool gauss_legendre_01(int o, double *xi, double *w) {
    q128 x[kMaxOrder], ww[kMaxOrder];
    if (!gauss_legendre_01_q(o, x, ww)) return false;
    for (int j = 0; j < o; ++j) { xi[j] = (double)x[j]; w[j] = (double)ww[j]; }
    return true;
}

// Polynomial helper: p(th) = sum_k c[k] th^k, fixed capacity.
struct PolyQ {
    q128 c[kMaxCoef + 2];
    PolyQ() { for (auto &x : c) x = 0; }
};

inline PolyQ poly_mul(const PolyQ &a, const PolyQ &b) {
    PolyQ r;
    for (int i = 0; i < kMaxCoef + 2; ++i)
        for (int k = 0; i + k < kMaxCoef + 2; ++k) r.c[i + k] += a.c[i] * b.c[k];
    return r;
}

// th^e * (1-th)^g
inline PolyQ poly_th_pow_times_one_minus_pow(int e, int g) {
    PolyQ one_minus; one_minus.c[0] = 1; one_minus.c[1] = -1;
    PolyQ r; r.c[0] = 1;
    for (int i = 0; i < g; ++i) r = poly_mul(r, one_minus);
    PolyQ s;
    for (int k = 0; k + e < kMaxCoef + 2; ++k) s.c[k + e] = r.c[k];
    return s;
}

inline q128 binom(int n, int k) {
    q128 v = 1;
    for (int i = 1; i <= k; ++i) v = v * (q128)(n - k + i) / (q128)i;
    return v;
}

// coef[(((mat*o + j)*o + l)*(2o) + k)*2 + {0,1}] = (hi, lo) double-double pair of the
// coefficient of th^k in A_jl (mat=0) / B_jl (mat=1): hi + lo carries 106 bits of the
// binary128 value, so that the device's double-double Horner gives A,B that are "rounded
// once" (D:O7).
inline std::vector<double> ab_polynomial_coefficients(int o) {
    q128 xi[kMaxOrder], w[kMaxOrder];
    gauss_legendre_01_q(o, xi, w);
    // monomial coefficients of l_j: product of (x - xi_m)/(xi_j - xi_m)
    q128 c[kMaxOrder][kMaxOrder];
    for (int j = 0; j < o; ++j) {
        q128 p[kMaxOrder + 1];
        for (auto &x : p) x = 0;
        p[0] = 1;
        int deg = 0;
        for (int m = 0; m < o; ++m) {
            if (m == j) continue;
            q128 d = xi[j] - xi[m];
            q128 q[kMaxOrder + 1];
            for (auto &x : q) x = 0;
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
    auto put = [&](size_t idx, q128 v) {
        double hi = (double)v;
        coef[idx * 2] = hi;
        coef[idx * 2 + 1] = (double)(v - (q128)hi);
    };
    for (int j = 0; j < o; ++j)
        for (int l = 0; l < o; ++l) {
            PolyQ PA, PB;
            for (int a = 0; a < o; ++a)
                for (int b = 0; b < o; ++b) {
                    q128 cc = c[j][a] * c[l][b];
                    for (int r = 0; r <= b; ++r) {
                        PolyQ t = poly_th_pow_times_one_minus_pow(b - r, a + r + 1);
                        q128 s = cc * binom(b, r) / (q128)(a + r + 1);
                        for (int k = 0; k < nc; ++k) PA.c[k] += s * t.c[k];
                    }
                    for (int r = 0; r <= a; ++r) {
                        PolyQ t = poly_th_pow_times_one_minus_pow(r + b + 1, a - r);
                        q128 s = cc * binom(a, r) / (q128)(r + b + 1);
                        for (int k = 0; k < nc; ++k) PB.c[k] += s * t.c[k];
                    }
                }
            for (int k = 0; k < nc; ++k) {
                put(((size_t)(0 * o + j) * o + l) * nc + k, PA.c[k] / w[j]);
                put(((size_t)(1 * o + j) * o + l) * nc + k, PB.c[k] / w[j]);
            }
            // theta = 0: A = I and B = 0 exactly (int_0^1 l_j l_l = w_j delta_jl because the o-point
            // rule is exact for degree 2o-2), so integer shifts move data bit-exactly (D:R3, P4).
            put(((size_t)(0 * o + j) * o + l) * nc, (j == l) ? (q128)1 : (q128)0);
            put(((size_t)(1 * o + j) * o + l) * nc, (q128)0);
        }
    return coef;
}

}  // namespace sldg
