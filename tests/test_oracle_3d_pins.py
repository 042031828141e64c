"""Pins for the oracle in THREE space / velocity dimensions and for its global sums (CPU only).

The d_x = 3 / d_v = 3 branches of oracle_poisson_E (mode decode), oracle_rho, oracle_moments,
oracle_diagnostics and oracle_step are pinned here against things the oracle does not compute itself:
analytic plane waves, closed forms of drifting Maxwellians, numpy contractions with the LIBRARY
Gauss-Legendre weights, SURVEY P9 for the config-5 state (electric energy 3/4 (eps/k)^2 (4 pi)^3 =
5.9532e-1), SURVEY P10 (Landau rate -0.1533 +- 2 % in 2+2 D), a 3+3 D run that must reduce to the
already pinned 1+1 D run, and exact (rational) summation for mass / l2 / momentum / kinetic energy.
Every asymmetric choice below (different cell counts, box lengths, mode numbers, drifts per
dimension) is there so that a transposed dimension, a wrong sign or a dropped factor fails."""
import math

import numpy as np
import pytest

from paper_1907_08316_b200 import workloads as W
from tests.test_oracle_physics_pins import fit_gamma
from tests.test_oracle_pins import np_gl01


def _weights(o, cells, lo, hi, d):
    _, w = np_gl01(o)
    return np.tile(w * (hi[d] - lo[d]) / cells[d], cells[d])


def _outer(parts):
    """prod_a parts[a][p_a], flat, index 0 fastest."""
    out = np.asarray(parts[0], dtype=np.float64)
    for p in parts[1:]:
        out = np.multiply.outer(np.asarray(p, dtype=np.float64), out).reshape(-1)
    return out


# ---------------------------------------------------------------- O5 in 3-D: plane waves (D:R6)

def test_poisson_3d_plane_waves(oracle):
    """-Lap phi = cos(k.x + c)  =>  E_a = k_a/|k|^2 sin(k.x + c): three different mode numbers (one
    negative), three different box lengths and cell counts, non-zero lower corners."""
    cells, o = (6, 8, 10), 2                    # M_a = floor((n_a - 1)/2) = 2, 3, 4
    lo, hi = (0.5, -1.0, 2.0), (0.5 + 2 * np.pi, 2.0, 7.5)
    g = oracle.Grid(3, 1, cells + (1,), o, lo + (0.0,), hi + (1.0,))
    x = [g.coords(a) for a in range(3)]
    L = [hi[a] - lo[a] for a in range(3)]

    def wave(modes, c):
        k = [2 * np.pi * modes[a] / L[a] for a in range(3)]
        ph = (k[0] * x[0][None, None, :] + k[1] * x[1][None, :, None] + k[2] * x[2][:, None, None] + c).reshape(-1)
        kk = sum(v * v for v in k)
        return np.cos(ph), [k[a] / kk * np.sin(ph) for a in range(3)]

    rhs1, E1 = wave((1, -3, 4), 0.3)            # the highest kept mode in x_2 and x_3
    E = g.poisson_E(rhs1 - 1.0)
    for a in range(3):
        assert np.allclose(E[a], E1[a], rtol=0, atol=1e-13), a
    # superposition of two different waves (decode of every mode index, linearity) and a constant (R13)
    rhs2, E2 = wave((-2, 1, 0), -1.1)
    E = g.poisson_E(rhs1 + 0.25 * rhs2 + 3.0)
    for a in range(3):
        assert np.allclose(E[a], E1[a] + 0.25 * E2[a], rtol=0, atol=1e-13), a
    # a wave along one axis only leaves the other components zero
    _, E3 = wave((0, 2, 0), 0.0)
    E = g.poisson_E(wave((0, 2, 0), 0.0)[0] - 1.0)
    assert np.max(np.abs(E[0])) < 1e-14 and np.max(np.abs(E[2])) < 1e-14
    assert np.allclose(E[1], E3[1], rtol=0, atol=1e-13)


# ---------------------------------------------------------------- O4 / R12 with d_v = 3

@pytest.mark.parametrize("dx,cells", [(1, (3, 4, 5, 3)), (2, (3, 2, 4, 3, 5)), (3, (2, 3, 2, 4, 3, 2))])
def test_rho_with_three_velocity_dimensions_vs_numpy(oracle, dx, cells):
    o, dv = 3, 3
    lo = (0.0,) * dx + (-4.0, -3.0, -5.0)
    hi = tuple(1.0 + a for a in range(dx)) + (4.5, 3.5, 4.0)
    g = oracle.Grid(dx, dv, cells, o, lo, hi)
    rng = np.random.default_rng(7 + dx)
    f = rng.uniform(-1.0, 1.0, g.ndof)
    Wv = _outer([_weights(o, cells, lo, hi, dx + a) for a in range(dv)])     # v_1 fastest
    V = Wv.size
    ref = -np.einsum("v,vx->x", Wv, f.reshape(V, g.X))
    assert np.allclose(g.rho(f), ref, rtol=0, atol=1e-13)
    f32 = f.astype(np.float32)
    ref32 = -np.einsum("v,vx->x", Wv, f32.astype(np.float64).reshape(V, g.X))
    assert np.allclose(g.rho(f32), ref32, rtol=0, atol=1e-13)


def test_drifting_maxwellian_3v_closed_forms(oracle):
    """rho = -1, P = u |Omega_x|, K = (3 + |u|^2) |Omega_x| / 2 for a unit-density Maxwellian with drift
    u = (0.7, -1.1, 0.4): distinct drifts and boxes per v-dimension catch swapped components."""
    u = (0.7, -1.1, 0.4)
    cells, o = (2, 3, 26, 28, 24), 3
    lo, hi = (0.0, 1.0, -8.0, -10.0, -8.5), (1.5, 3.0, 9.0, 8.0, 9.5)
    g = oracle.Grid(2, 3, cells, o, lo, hi)
    c = [g.coords(d) for d in range(5)]
    gv = _outer([np.exp(-0.5 * (c[2 + a] - u[a]) ** 2) / np.sqrt(2 * np.pi) for a in range(3)])
    f = np.multiply.outer(gv, np.ones(g.X)).reshape(-1)
    area = 1.5 * 2.0
    assert np.allclose(g.rho(f), -1.0, rtol=0, atol=1e-9)
    P, K = g.moments(f)
    assert np.allclose(P, np.array(u) * area, rtol=0, atol=1e-8)
    assert abs(K - 0.5 * (3 + sum(x * x for x in u)) * area) < 1e-8
    mass, l2, _ = g.diagnostics(f)
    assert abs(mass - area) < 1e-8
    # int M^2 dv = (4 pi)^{-3/2} for a unit Maxwellian in 3 v-dimensions
    assert abs(l2 ** 2 - area * (4 * np.pi) ** -1.5) < 1e-9


# ---------------------------------------------------------------- R12: the global sums against exact summation

def _exact_sums(f, Wv, Wx, va=None, v2=None):
    """sum_g Wv Wx f (and the other invariants) in exact rational arithmetic on the given doubles."""
    from fractions import Fraction as Fr
    V, X = Wv.size, Wx.size
    fv = f.reshape(V, X)
    m = s2 = k = Fr(0)
    p = [Fr(0)] * (0 if va is None else va.shape[0])
    for v in range(V):
        wv = Fr(float(Wv[v]))
        row_m = sum((Fr(float(Wx[x])) * Fr(float(fv[v, x])) for x in range(X)), Fr(0))
        m += wv * row_m
        s2 += wv * sum((Fr(float(Wx[x])) * Fr(float(fv[v, x])) ** 2 for x in range(X)), Fr(0))
        if va is not None:
            for a in range(len(p)):
                p[a] += Fr(float(va[a, v])) * wv * row_m
            k += Fr(float(v2[v])) * wv * row_m
    return m, s2, p, k


@pytest.mark.parametrize("dx,dv,cells,dtype", [(1, 1, (9, 40), np.float64), (2, 2, (3, 4, 5, 6), np.float64),
                                               (2, 3, (2, 3, 3, 4, 2), np.float32), (3, 3, (2, 2, 3, 3, 2, 2), np.float64)])
def test_global_sums_are_the_exact_sums_rounded(oracle, dx, dv, cells, dtype):
    """mass, l2, momentum and kinetic energy are single sums over all nodes (R12); the oracle's long-double
    accumulation must give the exactly summed value to a few ulp -- it owes its accuracy to the extended
    accumulator, not to a particular grouping of the terms.  Mixed-sign f makes the sums cancel."""
    o = 2
    lo = (0.0,) * dx + (-4.0, -3.0, -5.0)[:dv]
    hi = tuple(1.0 + 0.5 * a for a in range(dx)) + (4.5, 3.5, 4.0)[:dv]
    g = oracle.Grid(dx, dv, cells, o, lo, hi)
    rng = np.random.default_rng(1)
    f = (rng.uniform(-1.0, 1.0, g.ndof) * 10.0 ** rng.uniform(-6, 0, g.ndof)).astype(dtype)
    # the weights as the definition has them, W = prod_d h_d w_jd, from the oracle's own rule and nodes
    # (this test pins the SUMMATION; the rule and the weight products are pinned elsewhere)
    xi, w = oracle.gauss_legendre(o)

    def wts(d):
        return np.tile(w * ((hi[d] - lo[d]) / cells[d]), cells[d])

    def prod_left_to_right(parts):          # ((1 * a_0) * a_1) * ... per node, the order the definition is coded in
        out = np.ones(1)
        for a, p in enumerate(parts):
            out = (out[None, :] if a else out) * (p[:, None] if a else p)
            out = out.reshape(-1)
        return out
    Wx = prod_left_to_right([wts(d) for d in range(dx)])
    Wv = prod_left_to_right([wts(dx + a) for a in range(dv)])
    cv = [g.coords(dx + a) for a in range(dv)]
    Nv = [cells[dx + a] * o for a in range(dv)]
    idx = np.unravel_index(np.arange(Wv.size), tuple(reversed(Nv)))
    va = np.array([cv[a][idx[dv - 1 - a]] for a in range(dv)])
    v2 = np.zeros(Wv.size)
    for a in range(dv):
        v2 = v2 + va[a] * va[a]
    m, s2, p, k = _exact_sums(f.astype(np.float64), Wv, Wx, va, v2)
    mass, l2, _ = g.diagnostics(f)
    P, K = g.moments(f)
    scale_m = float(sum(abs(float(x)) for x in (Wv[:, None] * Wx[None, :] * np.abs(f.astype(np.float64)).reshape(Wv.size, Wx.size)).reshape(-1)))
    ulp = np.spacing
    # |error| <= 2 ulp of the result + 1e-19 of the sum of |terms| (long double accumulation)
    assert abs(mass - float(m)) <= 2 * ulp(abs(float(m))) + 1e-18 * scale_m
    assert abs(l2 - math.sqrt(float(s2))) <= 2 * ulp(l2)
    for a in range(dv):
        assert abs(P[a] - float(p[a])) <= 2 * ulp(abs(float(p[a]))) + 1e-17 * scale_m, a
    assert abs(K - 0.5 * float(k)) <= 2 * ulp(abs(0.5 * float(k))) + 1e-17 * scale_m


@pytest.mark.parametrize("dx,dv,cells,dtype", [(1, 1, (5, 300), np.float64), (2, 2, (2, 3, 20, 24), np.float64),
                                               (1, 3, (3, 8, 6, 10), np.float32), (3, 3, (1, 2, 1, 6, 5, 7), np.float64)])
def test_rho_is_the_exact_sum_rounded(oracle, dx, dv, cells, dtype):
    """O4: rho[x] = -sum_v W_v f[v][x] is a sum with no order.  The oracle's long-double running sum
    must give the exactly summed value (rational arithmetic on the same doubles) to 1 ulp -- with mixed-sign
    terms spanning six decades, where a double running sum over the same V terms is visibly off."""
    from fractions import Fraction as Fr
    o = 2
    lo = (0.0,) * dx + (-4.0, -3.0, -5.0)[:dv]
    hi = tuple(1.0 + 0.5 * a for a in range(dx)) + (4.5, 3.5, 4.0)[:dv]
    g = oracle.Grid(dx, dv, cells, o, lo, hi)
    rng = np.random.default_rng(7)
    f = (rng.uniform(-1.0, 1.0, g.ndof) * 10.0 ** rng.uniform(-6, 0, g.ndof)).astype(dtype)
    xi, w = oracle.gauss_legendre(o)
    Wv = np.ones(1)
    for a in range(dv):                       # ((1 * W_1) * W_2) * W_3 per node, v_1 fastest
        wa = np.tile(w * ((hi[dx + a] - lo[dx + a]) / cells[dx + a]), cells[dx + a])
        Wv = (Wv[None, :] * wa[:, None]).reshape(-1)
    V, X = Wv.size, g.X
    fv = f.astype(np.float64).reshape(V, X)
    rho = g.rho(f)
    worst_naive = 0.0
    for x in range(X):
        exact = -sum((Fr(float(Wv[v])) * Fr(float(fv[v, x])) for v in range(V)), Fr(0))
        scale = float(np.sum(np.abs(Wv * fv[:, x])))
        assert abs(Fr(float(rho[x])) - exact) <= Fr(float(np.spacing(abs(float(exact))))) + Fr(scale) * Fr(1, 10 ** 18), x
        naive = 0.0
        for v in range(V):
            naive += Wv[v] * fv[v, x]
        worst_naive = max(worst_naive, abs(float(Fr(-naive) - exact)) / scale)
    if V >= 1000:
        assert worst_naive > 2e-17           # the double running sum really is worse (what the oracle avoids)


# ---------------------------------------------------------------- P9 for the config-5 state (3+3 D)

def test_P9_initial_field_of_the_3p3_landau_state(oracle):
    """E_a = -(eps/k) sin(k x_a) for each a; electric energy = 3 * 1/4 (eps/k)^2 (4 pi)^3 = 5.9532e-1
     on a reduced grid with a different cell count per x-dimension."""
    cfg = W.CONFIG5.scaled((8, 6, 10, 14, 12, 16))
    g = oracle.Grid(cfg.dx, cfg.dv, cfg.cells, cfg.order, cfg.lo, cfg.hi)
    coords = [g.coords(d) for d in range(6)]
    f = W.initial_state(cfg, coords)
    E = g.poisson_E(g.rho(f))
    amp = cfg.eps / cfg.k
    N = cfg.N
    shape = (N[2], N[1], N[0])
    for a in range(3):
        s = -amp * np.sin(cfg.k * coords[a])
        ref = np.broadcast_to(s.reshape([-1 if (2 - b) == a else 1 for b in range(3)]), shape).reshape(-1)
        assert np.allclose(E[a], ref, rtol=0, atol=2e-6), a     # Maxwellian quadrature on 12-16 v-cells ~1e-5 relative
    mass, l2, ee = g.diagnostics(f)
    assert abs(ee / 5.9532e-1 - 1) < 2e-4
    assert abs(ee / (3 * 0.25 * amp ** 2 * (4 * np.pi) ** 3) - 1) < 2e-4
    assert abs(mass / (4 * np.pi) ** 3 - 1) < 1e-4


# ---------------------------------------------------------------- P10 in 2+2 D

def test_P10_landau_rate_2p2(oracle):
    """The k = 0.5 mode of each x-direction of the 2+2 D Landau state decays at gamma = -0.1533 +- 2 %
    (BASELINE.json north_star) on the reduced grid 16^2 x 32^2 cells."""
    cfg = W.CONFIG3.scaled((16, 16, 32, 32), steps=200)
    g = oracle.Grid(cfg.dx, cfg.dv, cfg.cells, cfg.order, cfg.lo, cfg.hi)
    f = W.initial_state(cfg, [g.coords(d) for d in range(4)])
    ee, mass = [], []
    for n in range(cfg.steps + 1):
        if n:
            g.step(f, cfg.dt)
        m, _, e = g.diagnostics(f)
        ee.append(e)
        mass.append(m)
    gamma, peaks = fit_gamma(np.array(ee), cfg.dt)
    assert abs(gamma / -0.1533 - 1) < 0.02
    assert abs(ee[0] / 3.1582734e-2 - 1) < 1e-6                                   # P9, config 3
    assert np.max(np.abs(np.array(mass) / mass[0] - 1)) < 1e-13                   # P5
    # the state is symmetric under x_1 <-> x_2: E_2(x_1, x_2) = E_1(x_2, x_1) up to the rounding of 200 steps
    E = g.poisson_E(g.rho(f))
    X1 = cfg.N[0]
    assert np.allclose(E[0].reshape(-1, X1), E[1].reshape(-1, X1).T, rtol=0, atol=1e-10 * np.max(np.abs(E)))


# ---------------------------------------------------------------- oracle_step in 3+3 D reduces to the 1+1 D run

@pytest.mark.parametrize("a", [0, 1, 2])
def test_3p3_step_reduces_to_the_1p1_run_along_each_axis(oracle, a):
    """A 3+3 D state that varies only in (x_a, v_a), times transverse factors that integrate to exactly 1
    on the grid, must evolve as the 1+1 D run (pinned by the Landau rate) times those factors: the other
    x-sweeps translate a constant, the other v-sweeps see E_b = 0.  Different cell counts and boxes per
    dimension: a mix-up of which E component drives which v-sweep, or of x_a <-> v_a pairing, fails."""
    o, steps, dt = 2, 15, 0.1
    nx1, nv1 = 16, 32
    cells_x = [2, 3, 2]; cells_v = [5, 4, 6]
    lo_x = [0.0, 1.0, -2.0]; hi_x = [3.0, 2.5, 1.0]
    lo_v = [-5.0, -4.5, -5.5]; hi_v = [5.5, 5.0, 4.5]
    cells_x[a], cells_v[a] = nx1, nv1
    lo_x[a], hi_x[a], lo_v[a], hi_v[a] = 0.0, 4 * np.pi, -6.0, 6.0
    g3 = oracle.Grid(3, 3, cells_x + cells_v, o, lo_x + lo_v, hi_x + hi_v)
    g1 = oracle.Grid(1, 1, (nx1, nv1), o, (0.0, -6.0), (4 * np.pi, 6.0))
    x, v = g1.coords(0), g1.coords(1)
    f1 = np.multiply.outer(np.exp(-0.5 * v * v) / np.sqrt(2 * np.pi), 1.0 + 0.05 * np.cos(0.5 * x)).reshape(-1)
    # transverse velocity factors normalised so that their Gauss sums are exactly 1 (then rho_3D = rho_1D)
    parts_x, parts_v = [], []
    for b in range(3):
        if b == a:
            parts_x.append(None); parts_v.append(None)
            continue
        parts_x.append(np.ones(cells_x[b] * o))
        cv = g3.coords(3 + b)
        gb = np.exp(-0.5 * cv * cv)
        wb = _weights(o, cells_x + cells_v, lo_x + lo_v, hi_x + hi_v, 3 + b)
        parts_v.append(gb / np.dot(wb, gb))
    N3 = [c * o for c in cells_x + cells_v]
    f1_2d = f1.reshape(nv1 * o, nx1 * o)               # [v_a][x_a]

    def embed(f1_2d):
        # f3[v3][v2][v1][x3][x2][x1]
        shp = [1] * 6
        out = np.ones(tuple(reversed(N3)))
        for b in range(3):
            if b == a:
                continue
            sx = [1] * 6; sx[5 - b] = N3[b]
            sv = [1] * 6; sv[5 - (3 + b)] = N3[3 + b]
            out = out * parts_x[b].reshape(sx) * parts_v[b].reshape(sv)
        s = [1] * 6; s[5 - a] = N3[a]; s[5 - (3 + a)] = N3[3 + a]
        return (out * f1_2d.reshape(s)).reshape(-1)

    f3 = embed(f1_2d)
    area = np.prod([hi_x[b] - lo_x[b] for b in range(3) if b != a])
    ee1, ee3 = [], []
    for n in range(steps):
        g1.step(f1, dt)
        g3.step(f3, dt)
        ee1.append(g1.diagnostics(f1)[2])
        ee3.append(g3.diagnostics(f3)[2])
    ref = embed(f1.reshape(nv1 * o, nx1 * o))
    assert np.max(np.abs(f3 - ref)) <= 1e-12 * np.max(np.abs(ref))
    assert np.allclose(np.array(ee3), area * np.array(ee1), rtol=1e-10, atol=0)
    E = g3.poisson_E(g3.rho(f3))
    for b in range(3):
        if b != a:
            assert np.max(np.abs(E[b])) < 1e-12 * np.max(np.abs(E[a]))
