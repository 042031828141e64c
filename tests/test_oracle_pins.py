"""Pins for the CPU oracle: the oracle is checked
against what the paper and the mathematics fix, never against itself or the CUDA path.

Independent routes used here: numpy's leggauss (library Gauss-Legendre rule), sympy
(exact symbolic integration with radicals), mpmath (adaptive quadrature, brute force),
closed forms typed from the derivation, and invariants the paper states (P:49 mass
conservation, P:65 L2 projection, P:224 Landau decay rate).
"""
import os

import numpy as np
import pytest

from paper_1907_08316_b200 import workloads as W

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def np_gl01(o):
    """Library Gauss-Legendre rule mapped to [0,1] (independent of the oracle's Newton)."""
    r, w = np.polynomial.legendre.leggauss(o)
    return 0.5 * (r + 1.0), 0.5 * w


# ---------------------------------------------------------------- O1: nodes and weights

@pytest.mark.parametrize("o", [1, 2, 3, 4, 5, 6])
def test_gauss_legendre_matches_library_and_is_exact(oracle, o):
    xi, w = oracle.gauss_legendre(o)
    xr, wr = np_gl01(o)
    assert np.allclose(xi, xr, rtol=0, atol=2e-16)
    assert np.allclose(w, wr, rtol=0, atol=4e-16)
    assert np.all(np.diff(xi) > 0) or o == 1
    for deg in range(2 * o):          # exact for monomials up to degree 2o-1 on [0,1]
        assert abs(np.dot(w, xi ** deg) - 1.0 / (deg + 1)) < 5e-16


def test_gauss_legendre_closed_forms(oracle):
    xi, w = oracle.gauss_legendre(2)
    assert np.allclose(xi, [0.5 - np.sqrt(3) / 6, 0.5 + np.sqrt(3) / 6], atol=1e-16)
    assert np.allclose(w, [0.5, 0.5], atol=1e-16)
    xi, w = oracle.gauss_legendre(3)
    assert np.allclose(xi, [0.5 - np.sqrt(15) / 10, 0.5, 0.5 + np.sqrt(15) / 10], atol=1e-16)
    assert np.allclose(w, [5 / 18, 8 / 18, 5 / 18], atol=1e-16)


def test_lagrange_is_cardinal(oracle):
    for o in (2, 3, 4):
        xi, _ = oracle.gauss_legendre(o)
        for j in range(o):
            for q in range(o):
                assert oracle.lagrange(o, xi, j, xi[q]) == (1.0 if j == q else 0.0)
        # partition of unity at an arbitrary point
        assert abs(sum(oracle.lagrange(o, xi, j, 0.3137) for j in range(o)) - 1.0) < 1e-15


def test_node_coords(oracle):
    c = oracle.node_coords(5, 3, -2.0, 3.0)
    xr, _ = np_gl01(3)
    ref = np.array([-2.0 + (i + xr[j]) * 1.0 for i in range(5) for j in range(3)])
    assert np.allclose(c, ref, atol=1e-15)


def test_shift_split(oracle):
    # R3: delta = -sigma, m = floor(delta) toward -inf, theta = delta - m in [0,1)
    assert oracle.shift_split(0.0) == (0, 0.0)
    assert oracle.shift_split(2.0) == (-2, 0.0)
    assert oracle.shift_split(-3.0) == (3, 0.0)
    assert oracle.shift_split(0.25) == (-1, 0.75)
    assert oracle.shift_split(-0.25) == (0, 0.25)
    assert oracle.shift_split(1.5) == (-2, 0.5)
    m, th = oracle.shift_split(-2.75)
    assert m == 2 and th == 0.75


# ---------------------------------------------------------------- O2: A(theta), B(theta)

def test_P1_order1_is_upwind(oracle):
    for th in (0.0, 0.1, 0.5, 0.9375):
        A, B = oracle.assemble_AB(1, th)
        assert abs(A[0, 0] - (1 - th)) < 1e-16 and abs(B[0, 0] - th) < 1e-16


def test_P2_order2_closed_form(oracle):
    s3 = np.sqrt(3.0)
    for th in np.linspace(0.0, 0.999, 38):
        A, B = oracle.assemble_AB(2, th)
        Ar = np.array([[1 - 2 * th + th ** 3, th * (1 + s3 - s3 * th - th ** 2)],
                       [th * (1 - s3 + s3 * th - th ** 2), 1 - 2 * th + th ** 3]])
        Br = np.array([[th * (-1 + 3 * th - th ** 2), th * (2 - s3 + (s3 - 3) * th + th ** 2)],
                       [th * (2 + s3 - (3 + s3) * th + th ** 2), th * (-1 + 3 * th - th ** 2)]])
        assert np.allclose(A, Ar, rtol=0, atol=2e-15)
        assert np.allclose(B, Br, rtol=0, atol=2e-15)


def test_P3_golden_values_theta_quarter(oracle):
    rows = np.loadtxt(os.path.join(GOLDEN, "ab_theta_quarter.txt"))
    for o in (2, 3):
        A, B = oracle.assemble_AB(o, 0.25)
        for r in rows[rows[:, 0] == o]:
            j, l = int(r[1]), int(r[2])
            assert abs(A[j, l] - r[3]) < 5e-16, (o, j, l)
            assert abs(B[j, l] - r[4]) < 5e-16, (o, j, l)


def _sympy_AB(o, theta):
    """Exact symbolic A,B: sympy Gauss-Legendre nodes as radicals, exact integration."""
    import sympy as sp
    x = sp.symbols("x")
    roots = sorted(sp.Poly(sp.legendre(o, x), x).all_roots(), key=lambda r: float(r))
    xi = [(1 + r) / 2 for r in roots]
    ell = [sp.prod([(x - xi[m]) / (xi[j] - xi[m]) for m in range(o) if m != j]) for j in range(o)]
    w = [sp.integrate(sp.expand(ell[j]), (x, 0, 1)) for j in range(o)]
    th = sp.nsimplify(theta)
    A = np.zeros((o, o))
    B = np.zeros((o, o))
    for j in range(o):
        for l in range(o):
            a = sp.integrate(sp.expand(ell[j] * ell[l].subs(x, x + th)), (x, 0, 1 - th)) / w[j]
            b = sp.integrate(sp.expand(ell[j] * ell[l].subs(x, x + th - 1)), (x, 1 - th, 1)) / w[j]
            A[j, l] = float(sp.N(a, 30))
            B[j, l] = float(sp.N(b, 30))
    return A, B


@pytest.mark.parametrize("o,theta", [(2, "1/4"), (3, "7/10")])
def test_P3_sympy_exact_integration(oracle, o, theta):
    A, B = oracle.assemble_AB(o, float(eval(theta.replace("/", "./"))))
    Ar, Br = _sympy_AB(o, theta)
    assert np.allclose(A, Ar, rtol=0, atol=2e-15)
    assert np.allclose(B, Br, rtol=0, atol=2e-15)


@pytest.mark.parametrize("o", [1, 2, 3, 4, 6])
def test_P4_theta_zero_is_identity_exactly(oracle, o):
    A, B = oracle.assemble_AB(o, 0.0)
    assert np.array_equal(A, np.eye(o))
    assert np.array_equal(B, np.zeros((o, o)))


@pytest.mark.parametrize("o", [1, 2, 3, 4, 5, 6])
def test_P5_P6_row_sums_mass_persymmetry(oracle, o):
    _, w = np_gl01(o)
    for th in (0.0, 1e-9, 0.123, 0.5, 0.77, 1 - 1e-9):
        A, B = oracle.assemble_AB(o, th)
        # constants preserved: sum_l (A+B)_jl = 1
        assert np.allclose((A + B).sum(axis=1), 1.0, rtol=0, atol=1e-14)
        # mass: sum_j w_j (A+B)_jl = w_l
        assert np.allclose(w @ (A + B), w, rtol=0, atol=1e-14)
        # persymmetry (reflection x -> -x): B_jl(theta) = A_{o-1-j,o-1-l}(1-theta)
        if 0.0 < th < 1.0:
            A1, _ = oracle.assemble_AB(o, 1.0 - th)
            assert np.allclose(B, A1[::-1, ::-1], rtol=0, atol=1e-13)


def test_assemble_rejects_theta_outside_unit_interval(oracle):
    with pytest.raises(ValueError):
        oracle.assemble_AB(2, 1.0)
    with pytest.raises(ValueError):
        oracle.assemble_AB(2, -0.1)


def test_R3_shift_split_never_returns_theta_one(oracle):
    """delta = -sigma a hair below an integer: fl(delta - floor(delta)) rounds to 1.0; R3 makes it
    the next integer shift with theta = 0 (the translation is continuous across integers)."""
    for s, m_exp in ((1e-20, 0), (1.0 + 1e-17, -1), (-3.0 + 1e-18, 3)):
        m, th = oracle.shift_split(s)
        assert 0.0 <= th < 1.0 and (m, th) == (m_exp, 0.0)
    assert oracle.shift_split(-1e-20) == (0, 1e-20)
    assert oracle.shift_split(-0.25) == (0, 0.25) and oracle.shift_split(0.25) == (-1, 0.75)
