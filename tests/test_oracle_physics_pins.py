"""Pins for the oracle's rho, Poisson, advect, step and diagnostics (O3..O6; P5, P8, P9, P10)."""
import math

import numpy as np
import pytest

from paper_1907_08316_b200 import workloads as W
from tests.test_oracle_pins import np_gl01


def _grid(oracle, cfg):
    g = oracle.Grid(cfg.dx, cfg.dv, cfg.cells, cfg.order, cfg.lo, cfg.hi)
    coords = [g.coords(d) for d in range(cfg.dx + cfg.dv)]
    return g, coords


def _np_weights(cfg, d):
    """Quadrature weight of every node of dimension d from the LIBRARY rule."""
    _, w = np_gl01(cfg.order)
    h = (cfg.hi[d] - cfg.lo[d]) / cfg.cells[d]
    return np.tile(w * h, cfg.cells[d])


# ---------------------------------------------------------------- O4: rho

def test_rho_is_minus_the_velocity_integral(oracle):
    cfg = W.CONFIG1.scaled((8, 32))
    g, coords = _grid(oracle, cfg)
    gx, gv = W.initial_factors(cfg, coords)
    f = W.initial_state(cfg, coords)
    rho = g.rho(f)
    # separable state: rho[x] = -gx[x] * sum_v W_v gv[v]  (library weights)
    ref = -gx * np.dot(_np_weights(cfg, 1), gv)
    assert np.allclose(rho, ref, rtol=0, atol=1e-15)
    # and the Maxwellian integrates to erf(6/sqrt 2) on [-6,6] (Gauss quadrature error ~1e-7 here)
    assert np.allclose(rho, -gx * math.erf(6 / math.sqrt(2)), rtol=0, atol=1e-6)


def test_rho_2d2v_and_f32(oracle):
    cfg = W.CONFIG3.scaled((4, 3, 6, 5))
    g, coords = _grid(oracle, cfg)
    rng = np.random.default_rng(3)
    f = rng.random(cfg.ndof)
    Wv = np.multiply.outer(_np_weights(cfg, 3), _np_weights(cfg, 2)).reshape(-1)
    ref = -(Wv[:, None] * f.reshape(cfg.V, cfg.X)).sum(axis=0)
    assert np.allclose(g.rho(f), ref, rtol=0, atol=1e-13)
    f32 = f.astype(np.float32)
    ref32 = -(Wv[:, None] * f32.astype(np.float64).reshape(cfg.V, cfg.X)).sum(axis=0)
    assert np.allclose(g.rho(f32), ref32, rtol=0, atol=1e-13)     # fp64 accumulators


# ---------------------------------------------------------------- O5: Poisson

def test_poisson_single_mode_1d(oracle):
    cfg = W.CONFIG1.scaled((16, 4))
    g, coords = _grid(oracle, cfg)
    x = coords[0]
    for mode in (1, 3, 7):                      # M = floor((16-1)/2) = 7 is the last kept mode
        k = 2 * np.pi * mode / (cfg.hi[0] - cfg.lo[0])
        # -phi'' = cos(kx + 0.3)  ->  E = -phi' = sin(kx + 0.3)/k ; rho = rhs - 1
        rho = np.cos(k * x + 0.3) - 1.0
        E = g.poisson_E(rho)[0]
        tol = 1e-13 if mode < 7 else 1e-5       # 2-point Gauss quadrature of the highest mode aliases
        assert np.allclose(E, np.sin(k * x + 0.3) / k, rtol=0, atol=tol), mode


def test_poisson_drops_mean_and_modes_at_or_above_cell_nyquist(oracle):
    cfg = W.CONFIG1.scaled((16, 4))
    g, coords = _grid(oracle, cfg)
    x = coords[0]
    L = cfg.hi[0] - cfg.lo[0]
    assert np.max(np.abs(g.poisson_E(np.full(x.size, 2.5))[0])) < 1e-14          # R13
    # cell Nyquist mode m = n/2 = 8 is not in the mode set |m| <= 7 (R6)
    k8 = 2 * np.pi * 8 / L
    E = g.poisson_E(np.cos(k8 * x) - 1.0)[0]
    assert np.max(np.abs(E)) < 0.05 * (1 / k8)


def test_poisson_2d_plane_wave_and_linearity(oracle):
    cfg = W.CONFIG3.scaled((8, 12, 2, 2))
    g, coords = _grid(oracle, cfg)
    x1, x2 = coords[0], coords[1]
    L1, L2 = cfg.hi[0] - cfg.lo[0], cfg.hi[1] - cfg.lo[1]
    k1, k2 = 2 * np.pi * 2 / L1, 2 * np.pi * (-3) / L2
    ph = k1 * x1[None, :] + k2 * x2[:, None]            # [x2][x1]: x1 fastest
    rho = (np.cos(ph) - 1.0).reshape(-1)
    E = g.poisson_E(rho)
    kk = k1 * k1 + k2 * k2
    assert np.allclose(E[0], (k1 / kk * np.sin(ph)).reshape(-1), rtol=0, atol=1e-13)
    assert np.allclose(E[1], (k2 / kk * np.sin(ph)).reshape(-1), rtol=0, atol=1e-13)
    rho_b = (0.3 * np.sin(2 * np.pi * x1 / L1)[None, :] * np.ones_like(x2)[:, None]).reshape(-1) - 1.0
    Eb = g.poisson_E(rho_b)
    Esum = g.poisson_E(rho + rho_b + 1.0)
    assert np.allclose(Esum, E + Eb, rtol=0, atol=1e-13)


def test_P9_initial_field_of_landau_state(oracle):
    # E = -(eps/k) sin(k x), electric energy = dx * 1/4 (eps/k)^2 |Omega_x| (v-truncation ~4e-9)
    cfg = W.CONFIG1
    g, coords = _grid(oracle, cfg)
    f = W.initial_state(cfg, coords)
    E = g.poisson_E(g.rho(f))[0]
    assert np.allclose(E, -(cfg.eps / cfg.k) * np.sin(cfg.k * coords[0]), rtol=0, atol=2e-10)
    mass, l2, ee = g.diagnostics(f)
    assert abs(ee - 1.2566370614359e-3) < 1e-10
    assert abs(ee / 1.25663705648e-3 - 1) < 1e-9        # S:P9, with the truncation
    assert abs(mass - 4 * np.pi * math.erf(6 / math.sqrt(2))) < 1e-6
    # l2^2 = int (1+eps cos)^2 dx * int M^2 dv = 4 pi (1 + eps^2/2) * erf(6)/(2 sqrt(pi))
    l2sq = 4 * np.pi * (1 + cfg.eps ** 2 / 2) * math.erf(6.0) / (2 * math.sqrt(np.pi))
    assert abs(l2 ** 2 - l2sq) < 1e-6


def test_P9_initial_field_2d2v(oracle):
    cfg = W.CONFIG3.scaled((16, 16, 16, 16))
    g, coords = _grid(oracle, cfg)
    f = W.initial_state(cfg, coords)
    E = g.poisson_E(g.rho(f))
    amp = cfg.eps / cfg.k
    E0 = (-amp * np.sin(cfg.k * coords[0])[None, :] * np.ones(cfg.N[1])[:, None]).reshape(-1)
    E1 = (-amp * np.sin(cfg.k * coords[1])[:, None] * np.ones(cfg.N[0])[None, :]).reshape(-1)
    assert np.allclose(E[0], E0, rtol=0, atol=1e-6)     # 16 v-cells: quadrature of the Maxwellian ~1e-7
    assert np.allclose(E[1], E1, rtol=0, atol=1e-6)
    _, _, ee = g.diagnostics(f)
    assert abs(ee / 3.1582734e-2 - 1) < 1e-5


# ---------------------------------------------------------------- O3: signs of the physics sweeps (R4)

def test_advect_x_moves_with_v(oracle):
    cfg = W.Config("t", 1, 1, (32, 4), 4, (0.0, -2.0), (2 * np.pi, 2.0))
    g, coords = _grid(oracle, cfg)
    x, v = coords
    f = (np.ones_like(v)[:, None] * np.sin(x)[None, :]).reshape(-1)
    tau = 0.37
    g.advect(f, 0, tau)
    ref = np.sin(x[None, :] - v[:, None] * tau).reshape(-1)       # f(x - v tau, v)
    assert np.max(np.abs(f - ref)) < 1e-6


def test_advect_v_moves_against_E(oracle):
    cfg = W.Config("t", 1, 1, (4, 32), 4, (0.0, -np.pi), (1.0, np.pi))
    g, coords = _grid(oracle, cfg)
    x, v = coords
    f = (np.sin(v)[:, None] * np.ones_like(x)[None, :]).reshape(-1)
    E = 0.5 + x                                                    # any E(x), one component
    tau = 0.21
    g.advect(f, 1, tau, E)
    ref = np.sin(v[:, None] + E[None, :] * tau).reshape(-1)       # f(x, v + E tau)
    assert np.max(np.abs(f - ref)) < 1e-6


# ---------------------------------------------------------------- O6: step, invariants, Landau rate

@pytest.fixture(scope="module")
def landau_trace(oracle):
    cfg = W.CONFIG1
    g, coords = _grid(oracle, cfg)
    f = W.initial_state(cfg, coords)
    tr = [g.diagnostics(f)]
    for _ in range(cfg.steps):
        g.step(f, cfg.dt)
        tr.append(g.diagnostics(f))
    return cfg, np.array(tr)


def fit_gamma(ee, dt):
    """R14: least squares through local maxima #2..#8 of a_n = 1/2 ln ee(t_n)."""
    a = 0.5 * np.log(ee)
    t = np.arange(a.size) * dt
    pk = [i for i in range(1, a.size - 1) if a[i] > a[i - 1] and a[i] > a[i + 1]]
    sel = pk[1:8]
    return np.polyfit(t[sel], a[sel], 1)[0], t[pk]


def test_P10_landau_damping_rate(landau_trace):
    cfg, tr = landau_trace
    gamma, peaks = fit_gamma(tr[:, 2], cfg.dt)
    assert abs(gamma / -0.1533 - 1) < 0.02                          # BASELINE.json north_star
    # oscillation frequency omega ~ 1.4156: energy peaks every pi/omega ~ 2.22
    assert abs(np.mean(np.diff(peaks[:8])) - np.pi / 1.4156) < 0.05


def test_P5_P8_step_conserves_mass_and_contracts_l2(landau_trace):
    _, tr = landau_trace
    assert np.max(np.abs(tr[:, 0] / tr[0, 0] - 1)) < 1e-13
    assert np.all(np.diff(tr[:, 1]) <= 1e-15)


def test_step_is_second_order_in_dt(oracle):
    # Strang splitting: halving dt reduces the splitting error ~4x (space error kept negligible)
    cfg = W.Config("t", 1, 1, (32, 64), 4, (0.0, -6.0), (4 * np.pi, 6.0), kind="landau", eps=0.05, k=0.5)
    g, coords = _grid(oracle, cfg)
    f0 = W.initial_state(cfg, coords)

    def run(nsteps):
        f = f0.copy()
        for _ in range(nsteps):
            g.step(f, 1.0 / nsteps)
        return f
    ref = run(32)
    e1 = np.max(np.abs(run(2) - ref))
    e2 = np.max(np.abs(run(4) - ref))
    assert 3.0 < e1 / e2 < 5.5


def test_f32_step_tracks_f64(oracle):
    cfg = W.CONFIG2.scaled((32, 32))
    g, coords = _grid(oracle, cfg)
    f64 = W.initial_state(cfg, coords)
    f32 = f64.astype(np.float32)
    for _ in range(20):
        g.step(f64, cfg.dt)
        g.step(f32, cfg.dt)
    assert f32.dtype == np.float32
    assert np.max(np.abs(f32 - f64)) < 2e-5 * np.max(np.abs(f64))
    m64, m32 = g.diagnostics(f64)[0], g.diagnostics(f32)[0]
    assert abs(m32 / m64 - 1) < 1e-6
