"""The oracle's A(theta), B(theta) against EXACT values for o = 1..6 (CPU only).

DESIGN.md O7 / R9 takes "A,B are assembled in fp64 and rounded once to T" literally: the matrices are
exact real numbers (integrals of polynomials with Gauss-Legendre nodes as roots) rounded once.  The
oracle reaches that by carrying out its o-point quadrature in long double (commit "Oracle: evaluate the
Gauss-Legendre rule and A,B in long double").  This file pins the claim on the CPU, by a route that
shares nothing with the oracle: 60-digit mpmath arithmetic on the monomial coefficients of the Lagrange
basis (Taylor shift, polynomial product, term-by-term antiderivative) -- no quadrature rule at all.

Statement pinned:  |oracle - exact| <= 1/2 ulp(exact) + 1e-18  for every entry, every theta tried,
including theta -> 0 and theta -> 1 where entries are tiny by cancellation.  The 1e-18 is the long-double
ABSOLUTE error of the O(1) terms an entry is summed from (measured <= 4.8e-19 at o = 6); for entries
>= 2^-6 in magnitude it is below half an ulp, i.e. those are within one ulp of the exact value."""
import numpy as np
import pytest

THETAS = [0.0, 2.0 ** -60, 1e-12, 1e-6, 1e-3, 0.25, 0.3, 0.5, 0.7, 0.875, 1 - 1e-3, 1 - 1e-6, 1 - 2.0 ** -40,
          1 - 2.0 ** -53] + list(np.random.default_rng(0).uniform(0, 1, 12))


def exact_AB(o, theta):
    """A, B as mpmath numbers (60 digits) from the definition, by exact polynomial algebra."""
    import mpmath as mp
    mp.mp.dps = 60
    if o == 1:
        r = [mp.mpf(0)]
    else:
        r = sorted(mp.findroot(lambda x: mp.legendre(o, x), mp.mpf(float(r0)), tol=mp.mpf("1e-110"), maxsteps=200)
                   for r0 in np.polynomial.legendre.leggauss(o)[0])
    xi = [(1 + x) / 2 for x in r]

    def polymul(a, b):
        c = [mp.mpf(0)] * (len(a) + len(b) - 1)
        for i, x in enumerate(a):
            for j, y in enumerate(b):
                c[i + j] += x * y
        return c

    def ell(j):                                  # ascending monomial coefficients of the Lagrange basis
        p = [mp.mpf(1)]
        for m in range(o):
            if m != j:
                p = polymul(p, [-xi[m] / (xi[j] - xi[m]), 1 / (xi[j] - xi[m])])
        return p

    def shifted(p, s):                           # coefficients of p(x + s)
        out = [mp.mpf(0)] * len(p)
        for k, c in enumerate(p):
            for i in range(k + 1):
                out[i] += c * mp.binomial(k, i) * s ** (k - i)
        return out

    def integral(p, a, b):
        return sum(c * (b ** (k + 1) - a ** (k + 1)) / (k + 1) for k, c in enumerate(p))

    L = [ell(j) for j in range(o)]
    w = [integral(L[j], 0, 1) for j in range(o)]
    th = mp.mpf(theta)
    A = [[integral(polymul(L[j], shifted(L[l], th)), 0, 1 - th) / w[j] for l in range(o)] for j in range(o)]
    B = [[integral(polymul(L[j], shifted(L[l], th - 1)), 1 - th, 1) / w[j] for l in range(o)] for j in range(o)]
    return A, B


@pytest.mark.parametrize("o", [1, 2, 3, 4, 5, 6])
def test_assemble_AB_is_the_exact_value_rounded_once(oracle, o):
    import mpmath as mp
    checked = within_one_ulp = 0
    for theta in THETAS:
        A, B = oracle.assemble_AB(o, theta)
        Ae, Be = exact_AB(o, theta)
        for got, exact in ((A, Ae), (B, Be)):
            for j in range(o):
                for l in range(o):
                    ex = exact[j][l]
                    if abs(ex) < mp.mpf("1e-45"):                  # exactly zero (theta = 0: A = I, B = 0)
                        assert got[j, l] == 0.0, (o, theta, j, l)
                        continue
                    err = abs(mp.mpf(float(got[j, l])) - ex)
                    half_ulp = mp.mpf(float(np.spacing(abs(float(ex))))) / 2
                    assert err <= half_ulp + mp.mpf("1e-18"), (o, theta, j, l, float(err))
                    checked += 1
                    if abs(ex) >= 2.0 ** -6:
                        assert err <= 2 * half_ulp, (o, theta, j, l, float(err))
                        within_one_ulp += 1
    assert checked >= 2 * o * o * (len(THETAS) - 1) and within_one_ulp > checked // 4


def test_exact_route_reproduces_the_printed_closed_form():
    """The exact route itself against SURVEY P2 (o = 2 closed form) so that it is not self-referential."""
    import mpmath as mp
    th = mp.mpf("0.3")
    s3 = mp.sqrt(3)
    A, B = exact_AB(2, 0.3)
    thd = mp.mpf(0.3)                            # the double 0.3, as exact_AB sees it
    assert abs(A[0][0] - (1 - 2 * thd + thd ** 3)) < mp.mpf("1e-50")
    assert abs(A[0][1] - thd * (1 + s3 - s3 * thd - thd ** 2)) < mp.mpf("1e-50")
    assert abs(B[1][0] - thd * (2 + s3 - (3 + s3) * thd + thd ** 2)) < mp.mpf("1e-50")
    assert abs(B[0][0] - thd * (-1 + 3 * thd - thd ** 2)) < mp.mpf("1e-50")
    assert th != thd
