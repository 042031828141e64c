"""Pins for the oracle's extra invariants (momentum, kinetic energy; S:8(f) NEXT-4, P:69/P:224/P:301)."""
import numpy as np

from paper_1907_08316_b200 import workloads as W


def test_shifted_maxwellian_closed_forms_1p1(oracle):
    # f = exp(-(v-u)^2/2)/sqrt(2 pi) on x in [0,L):  momentum = u L, kinetic = (1+u^2) L / 2
    L, u = 2.0, 1.3
    g = oracle.Grid(1, 1, (8, 64), 4, (0.0, -9.0), (L, 11.0))
    x, v = g.coords(0), g.coords(1)
    f = np.multiply.outer(np.exp(-0.5 * (v - u) ** 2) / np.sqrt(2 * np.pi), np.ones_like(x)).reshape(-1)
    P, K = g.moments(f)
    assert abs(P[0] - u * L) < 1e-12 and abs(K - 0.5 * (1 + u * u) * L) < 1e-12


def test_drifting_maxwellian_2p2_components_and_sign(oracle):
    # product Maxwellian with drift (u1, u2): P = (u1, u2) |Omega_x|, K = (2 + u1^2 + u2^2) |Omega_x| / 2.
    # distinct drifts and an asymmetric box catch swapped components, wrong sign, wrong weights.
    u1, u2 = 0.7, -1.1
    g = oracle.Grid(2, 2, (3, 2, 40, 44), 3, (0.0, 1.0, -8.0, -10.0), (1.5, 3.0, 9.0, 8.0))
    c = [g.coords(d) for d in range(4)]
    gv = np.multiply.outer(np.exp(-0.5 * (c[3] - u2) ** 2), np.exp(-0.5 * (c[2] - u1) ** 2)).reshape(-1) / (2 * np.pi)
    f = np.multiply.outer(gv, np.ones(g.X)).reshape(-1)
    P, K = g.moments(f)
    area = 1.5 * 2.0
    assert np.allclose(P, [u1 * area, u2 * area], rtol=0, atol=1e-10)
    assert abs(K - 0.5 * (2 + u1 * u1 + u2 * u2) * area) < 1e-10
    P32, K32 = g.moments(f.astype(np.float32))
    assert np.allclose(P32, P, rtol=1e-6) and abs(K32 - K) < 1e-6 * K


def test_polynomial_moments_are_exact(oracle):
    # o = 3: the rule integrates degree 5 exactly per cell; f = 1 + v (degree 1) times v^2 is degree 3.
    g = oracle.Grid(1, 1, (2, 5), 3, (0.0, -1.0), (1.0, 2.0))
    x, v = g.coords(0), g.coords(1)
    f = np.multiply.outer(1.0 + v, np.ones_like(x)).reshape(-1)
    P, K = g.moments(f)
    # int_{-1}^{2} v (1+v) dv = 3/2 + 3 = 4.5 ; 1/2 int v^2 (1+v) dv = 1/2 (3 + 15/4) = 3.375
    assert abs(P[0] - 4.5) < 1e-14 and abs(K - 3.375) < 1e-14


def test_landau_run_conserves_momentum_and_total_energy(oracle):
    # P:224 "mass and momentum conservation"; Fig. 15 tracks the total energy.
    cfg = W.CONFIG1.scaled((32, 32), steps=40)
    g = oracle.Grid(cfg.dx, cfg.dv, cfg.cells, cfg.order, cfg.lo, cfg.hi)
    f = W.initial_state(cfg, [g.coords(0), g.coords(1)])
    P0, K0 = g.moments(f)
    _, _, ee0 = g.diagnostics(f)
    for _ in range(cfg.steps):
        g.step(f, cfg.dt)
    P1, K1 = g.moments(f)
    _, _, ee1 = g.diagnostics(f)
    assert abs(P0[0]) < 1e-12 and abs(P1[0]) < 1e-9            # symmetric state: momentum stays ~0
    assert abs((K1 + ee1) - (K0 + ee0)) < 2e-5 * (K0 + ee0)    # total energy (not exactly conserved by splitting)
    assert abs(K1 - K0) > 10 * abs((K1 + ee1) - (K0 + ee0))    # while kinetic and electric energy do exchange
