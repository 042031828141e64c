"""CPU: the CUDA library's host-side tables (csrc/tables.hpp: closed-form Gauss-Legendre rule in
binary128, polynomial coefficients of A(theta), B(theta)) pinned WITHOUT a GPU and without the
oracle: against numpy's Gauss-Legendre rule and against exact integration (mpmath) of the
definition  A_jl = 1/w_j int_0^{1-th} l_j(x) l_l(x+th) dx,  B_jl = 1/w_j int_{1-th}^1 l_j(x) l_l(x+th-1) dx."""
import os
import subprocess

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def tables(tmp_path_factory):
    exe = str(tmp_path_factory.mktemp("tab") / "dump_tables")
    subprocess.run(["g++", "-std=c++17", "-O1", "-o", exe, os.path.join(ROOT, "tests", "host", "dump_tables.cpp")],
                   check=True)
    out = subprocess.run([exe], check=True, capture_output=True, text=True).stdout
    gl, ab = {}, {}
    for line in out.splitlines():
        p = line.split()
        o = int(p[1])
        vals = np.array([float(x) for x in p[2:]])
        if p[0] == "GL":
            gl[o] = (vals[0::2], vals[1::2])
        else:
            ab[o] = vals.reshape(2, o, o, 2 * o, 2)       # [mat][j][l][k][hi,lo]
    return gl, ab


@pytest.mark.parametrize("o", [1, 2, 3, 4, 5, 6])
def test_gauss_legendre_closed_forms_match_numpy(tables, o):
    xi, w = tables[0][o]
    r, W = np.polynomial.legendre.leggauss(o)
    assert np.max(np.abs(xi - 0.5 * (1 + r))) < 3e-16 and np.max(np.abs(w - 0.5 * W)) < 3e-16
    assert abs(w.sum() - 1.0) < 1e-15 and np.all(np.diff(xi) > 0)


@pytest.mark.parametrize("o", [1, 2, 3, 4, 5, 6])
def test_ab_polynomials_match_exact_integration(tables, o):
    import mpmath as mp
    mp.mp.dps = 40
    coef = tables[1][o]
    # roots of P_o to 40 digits: Newton (mpmath) on the Legendre polynomial from numpy's double roots
    r = sorted(mp.findroot(lambda x: mp.legendre(o, x), mp.mpf(float(r0)), tol=mp.mpf("1e-70"), maxsteps=100)
               for r0 in np.polynomial.legendre.leggauss(o)[0])
    xi = [(1 + x) / 2 for x in r]

    def ell(j, x):
        v = mp.mpf(1)
        for m in range(o):
            if m != j:
                v *= (x - xi[m]) / (xi[j] - xi[m])
        return v

    wq = [mp.quad(lambda x, j=j: ell(j, x), [0, 1]) for j in range(o)]
    for th in (mp.mpf("0.3"), mp.mpf("0.875")):
        for j in range(o):
            for l in range(o):
                A = mp.quad(lambda x: ell(j, x) * ell(l, x + th), [0, 1 - th]) / wq[j]
                B = mp.quad(lambda x: ell(j, x) * ell(l, x + th - 1), [1 - th, 1]) / wq[j]
                for mat, exact in ((0, A), (1, B)):
                    c = coef[mat, j, l]
                    val = sum((mp.mpf(float(c[k, 0])) + mp.mpf(float(c[k, 1]))) * th ** k for k in range(2 * o))
                    assert abs(val - exact) < mp.mpf("1e-25"), (o, mat, j, l)


@pytest.mark.parametrize("o", [1, 2, 3, 4, 5, 6])
def test_theta_zero_terms_are_exact(tables, o):
    coef = tables[1][o]
    for j in range(o):
        for l in range(o):
            assert coef[0, j, l, 0, 0] == (1.0 if j == l else 0.0) and coef[0, j, l, 0, 1] == 0.0
            assert coef[1, j, l, 0, 0] == 0.0 and coef[1, j, l, 0, 1] == 0.0
