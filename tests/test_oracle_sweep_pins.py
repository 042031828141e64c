"""Pins for the oracle's sweep (O2/O3/O7): P4, P5, P7, P8, P11, P12, P13 of SURVEY.md 8(c)."""
import numpy as np
import pytest

from tests.test_oracle_pins import np_gl01


def _line_matrices(oracle, o, sigma, dtype=np.float64):
    m, th = oracle.shift_split(sigma)
    A, B = oracle.assemble_AB(o, th)
    return m, A.astype(dtype), B.astype(dtype)


# ---------------------------------------------------------------- P4: integer shifts are exact

@pytest.mark.parametrize("dtype", [np.float64, np.float32])
@pytest.mark.parametrize("o", [1, 2, 3, 4, 5, 6])
def test_P4_integer_shift_is_a_bit_exact_roll(oracle, o, dtype):
    rng = np.random.default_rng(1)
    n = 7
    u = rng.standard_normal(n * o).astype(dtype)
    for s in (-9, -1, 0, 1, 2, 7, 15):
        m, A, B = _line_matrices(oracle, o, float(s), dtype)
        un = oracle.translate_line(o, A, B, m, u)
        # new(x) = old(x - s h): cell i takes the values of cell i - s
        assert np.array_equal(un.reshape(n, o), np.roll(u.reshape(n, o), s, axis=0))


def test_P4_integer_shift_multi_dimensional(oracle):
    rng = np.random.default_rng(2)
    N = np.array([6, 4, 9])          # o = 3 along dim 0 and 2, dim 1 has 4 nodes (o irrelevant there)
    o = 3
    f = rng.standard_normal(int(np.prod(N)))
    # sweep along dim 2 (3 cells), integer shift depending on the dim-0 node
    sigma = np.array([0.0, 1.0, 2.0, -1.0, 3.0, -4.0])
    g = oracle.translate(f.copy(), N, o, 2, sigma, [0])
    F = f.reshape(9, 4, 6)            # C order: dim 2 slowest
    G = g.reshape(9, 4, 6)
    for p0 in range(6):
        ref = np.roll(F[:, :, p0].reshape(3, 3, 4), int(sigma[p0]), axis=0).reshape(9, 4)
        assert np.array_equal(G[:, :, p0], ref)


# ---------------------------------------------------------------- P11: brute force on tiny input

def _brute_force_line(o, n, sigma, u):
    """L2 projection of the exactly translated piecewise polynomial, by adaptive quadrature
    (mpmath) with library nodes; no A/B matrices, no split into m and theta."""
    import mpmath as mp
    mp.mp.dps = 30
    xi, w = np_gl01(o)
    xi = [mp.mpf(float(x)) for x in xi]

    def ell(j, x):
        v = mp.mpf(1)
        for m in range(o):
            if m != j:
                v *= (x - xi[m]) / (xi[j] - xi[m])
        return v

    def u_old(x):                       # x in cell widths, periodic
        x = x - n * mp.floor(x / n)
        i = int(mp.floor(x))
        if i == n:
            i = n - 1
        return sum(mp.mpf(float(u[i * o + l])) * ell(l, x - i) for l in range(o))

    out = np.zeros(n * o)
    sig = mp.mpf(sigma)
    for i in range(n):
        # the translated function has a kink where x - sigma crosses a cell interface
        brk = sig - mp.floor(sig)
        pts = [mp.mpf(0), brk, mp.mpf(1)] if 0 < brk < 1 else [mp.mpf(0), mp.mpf(1)]
        for j in range(o):
            val = mp.quad(lambda s: ell(j, s) * u_old(i + s - sig), pts)
            out[i * o + j] = float(val / mp.mpf(float(w[j])))
    return out


@pytest.mark.parametrize("o,sigma", [(2, 0.3), (2, -1.6), (3, 0.45), (3, -0.2), (4, 2.25), (5, 0.37), (6, -0.7)])
def test_P11_brute_force_projection(oracle, o, sigma):
    rng = np.random.default_rng(o * 100 + 7)
    n = 4
    u = rng.standard_normal(n * o)
    m, A, B = _line_matrices(oracle, o, sigma)
    un = oracle.translate_line(o, A, B, m, u)
    ref = _brute_force_line(o, n, sigma, u)
    assert np.allclose(un, ref, rtol=0, atol=5e-14)


# ---------------------------------------------------------------- P7: polynomial reproduction

@pytest.mark.parametrize("o", [2, 3, 4, 5, 6])
def test_P7_polynomials_below_order_are_reproduced(oracle, o):
    n = 16
    xr, _ = np_gl01(o)
    x = (np.arange(n)[:, None] + xr[None, :]).reshape(-1)       # node coordinates in cell widths
    sigma = 2.37
    m, A, B = _line_matrices(oracle, o, sigma)
    interior = (x > 4) & (x < n - 1)                            # away from the periodic seam
    for deg in range(o):
        u = (x / n) ** deg
        un = oracle.translate_line(o, A, B, m, u)
        ref = ((x - sigma) / n) ** deg
        assert np.max(np.abs(un - ref)[interior]) < 5e-15, deg
    # degree o is NOT reproduced (the method is of order o, not more)
    u = (x / n) ** o
    un = oracle.translate_line(o, A, B, m, u)
    err = np.max(np.abs(un - ((x - sigma) / n) ** o)[interior])
    assert 1e-12 < err < 1e-2          # (1.4e-11 at o = 6 on 16 cells; round-off is 5e-15)


def test_sign_of_the_shift(oracle):
    # new(x) = old(x - sigma h): a bump moves to the RIGHT for sigma > 0 (R3)
    o, n = 3, 32
    xr, _ = np_gl01(o)
    x = (np.arange(n)[:, None] + xr[None, :]).reshape(-1)
    u = np.exp(-0.5 * ((x - 10.0) / 2.5) ** 2)
    m, A, B = _line_matrices(oracle, o, 4.5)
    un = oracle.translate_line(o, A, B, m, u)
    assert abs(x[np.argmax(un)] - 14.5) < 0.5
    assert np.max(np.abs(un - np.exp(-0.5 * ((x - 14.5) / 2.5) ** 2))) < 5e-4


# ---------------------------------------------------------------- P5 / P8: mass and L2

@pytest.mark.parametrize("dtype,tol", [(np.float64, 2e-15), (np.float32, 2e-7)])
@pytest.mark.parametrize("o", [2, 3, 4, 5, 6])
def test_P5_P8_mass_conserved_l2_contracts(oracle, o, dtype, tol):
    rng = np.random.default_rng(5)
    n = 24
    _, w = np_gl01(o)
    Wn = np.tile(w, n)
    u = rng.random(n * o).astype(dtype)
    mass0 = float(np.dot(Wn, u.astype(np.float64)))
    l2_prev = float(np.dot(Wn, u.astype(np.float64) ** 2))
    for sigma in (0.1, -0.73, 3.999, -5.5, 0.5):
        m, A, B = _line_matrices(oracle, o, sigma, dtype)
        u = oracle.translate_line(o, A, B, m, u)
        mass = float(np.dot(Wn, u.astype(np.float64)))
        l2 = float(np.dot(Wn, u.astype(np.float64) ** 2))
        assert abs(mass - mass0) <= tol * n * abs(mass0)
        assert l2 <= l2_prev * (1 + 10 * tol)
        l2_prev = l2


# ---------------------------------------------------------------- P12 / P13: dimension independence

def _grid_nd(rng, N):
    return rng.random(int(np.prod(N)))


@pytest.mark.parametrize("k", [0, 1, 2, 3])
def test_P12_nd_sweep_equals_1d_rule_on_every_line(oracle, k):
    rng = np.random.default_rng(11 + k)
    o = 2
    N = np.array([6, 4, 8, 6])
    f = _grid_nd(rng, N)
    # x-type dependence: shift depends on one other dimension; v-type: on two other dimensions
    dep = [d for d in range(4) if d != k][:2] if k >= 2 else [(k + 2) % 4]
    dep = sorted(dep)
    cnt = int(np.prod(N[dep]))
    sigma = rng.uniform(-3.5, 3.5, cnt)
    g = oracle.translate(f.copy(), N, o, k, sigma, dep)
    F = f.reshape(tuple(N[::-1]))     # axes reversed: axis (3-d) <-> dimension d
    G = g.reshape(tuple(N[::-1]))
    ax = 3 - k
    Fm = np.moveaxis(F, ax, -1)
    Gm = np.moveaxis(G, ax, -1)
    other = [d for d in range(4) if d != k][::-1]      # dimension of each remaining axis (slow -> fast)
    for idx in np.ndindex(Fm.shape[:-1]):
        p = {d: idx[a] for a, d in enumerate(other)}
        q, stride = 0, 1
        for d in dep:
            q += p[d] * stride
            stride *= N[d]
        m, A, B = _line_matrices(oracle, o, sigma[q])
        ref = oracle.translate_line(o, A, B, m, np.ascontiguousarray(Fm[idx]))
        assert np.array_equal(Gm[idx], ref)


def test_P13_sweeps_along_different_x_commute(oracle):
    rng = np.random.default_rng(21)
    o = 2
    N = np.array([8, 6, 4, 6])
    f = _grid_nd(rng, N)
    s0 = rng.uniform(-2, 2, N[2])     # x_1 shift depends on the v_1 node
    s1 = rng.uniform(-2, 2, N[3])     # x_2 shift depends on the v_2 node
    a = oracle.translate(oracle.translate(f.copy(), N, o, 0, s0, [2]), N, o, 1, s1, [3])
    b = oracle.translate(oracle.translate(f.copy(), N, o, 1, s1, [3]), N, o, 0, s0, [2])
    assert np.allclose(a, b, rtol=0, atol=1e-14)
    assert np.max(np.abs(a - f)) > 1e-2


def test_translate_rejects_bad_arguments(oracle):
    f = np.zeros(24)
    with pytest.raises(ValueError):
        oracle.translate(f, np.array([6, 4]), 2, 0, np.zeros(6), [0])     # dep == k
    with pytest.raises(ValueError):
        oracle.translate(f, np.array([6, 4]), 4, 0, np.zeros(4), [1])     # N_k not a multiple of o
