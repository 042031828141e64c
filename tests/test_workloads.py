"""The seeded input generators (paper_1907_08316_b200/workloads.py): sizes, determinism, recipe."""
import numpy as np

from paper_1907_08316_b200 import workloads as W


def test_config_sizes_match_baseline_json():
    # SURVEY.md section 8 size table / BASELINE.json configs
    assert W.CONFIG1.N == (128, 128) and W.CONFIG1.ndof == 16384
    assert W.CONFIG2.N == (768, 768) and W.CONFIG2.ndof == 589824
    assert W.CONFIG3.ndof == 128 ** 4 == 268435456
    assert W.CONFIG4.N == (384, 384, 192, 192) and W.CONFIG4.ndof == 5435817984
    assert W.CONFIG4.X == 147456
    assert W.CONFIG5.ndof == 4096000000 and W.CONFIG5.X == 64000
    assert W.CONFIG4.hi == (128.0, 128.0, 64.0, 64.0)              # unit cells


def test_uniform_generator_is_stateless_and_uniform():
    g = np.arange(200000, dtype=np.uint64)
    u = W.uniform(W.SEED, W.TAG_F, g)
    assert u.dtype == np.float64 and u.min() >= 0.0 and u.max() < 1.0
    assert abs(u.mean() - 0.5) < 3e-3 and abs(u.var() - 1 / 12) < 2e-3
    # stateless: any subset reproduces the same numbers
    assert np.array_equal(W.uniform(W.SEED, W.TAG_F, g[1234:1300]), u[1234:1300])
    # different tag / seed -> different stream
    assert not np.array_equal(W.uniform(W.SEED, W.TAG_F + 1, g[:64]), u[:64])
    assert not np.array_equal(W.uniform(W.SEED + 1, W.TAG_F, g[:64]), u[:64])
    # neighbouring counters are uncorrelated
    assert abs(np.corrcoef(u[:-1], u[1:])[0, 1]) < 0.01


def test_mix64_reference_vector():
    # splitmix64 finaliser of x = g + golden*(tag+1) + C*seed, worked by hand with Python ints
    def ref(seed, tag, g):
        M = (1 << 64) - 1
        x = (g + 0x9E3779B97F4A7C15 * (tag + 1) + 0xD1B54A32D192ED03 * seed) & M
        x ^= x >> 30
        x = (x * 0xBF58476D1CE4E5B9) & M
        x ^= x >> 27
        x = (x * 0x94D049BB133111EB) & M
        x ^= x >> 31
        return x
    for seed, tag, g in [(0, 0, 0), (W.SEED, 0, 1), (W.SEED, 17, 5435817983), (7, 3, 2 ** 40 + 11)]:
        assert int(W.mix64(seed, tag, np.array([g], dtype=np.uint64))[0]) == ref(seed, tag, g)


def test_config4_shift_tables():
    cfg = W.CONFIG4.scaled((4, 6, 5, 3))
    o = cfg.order
    sx = W.config4_shifts(cfg, 0)           # x_1 sweep: per cell of v_1, replicated to o nodes
    assert sx.shape == (cfg.N[2],)
    assert np.all(np.abs(sx) <= 3.5)
    assert np.array_equal(sx.reshape(-1, o), np.repeat(sx[::o, None], o, axis=1))
    sv = W.config4_shifts(cfg, 3)           # v_2 sweep: per x-cell (i_1, i_2)
    assert sv.shape == (cfg.X,)
    S = sv.reshape(cfg.N[1], cfg.N[0])
    cells = S[::o, ::o]
    assert np.array_equal(S, np.repeat(np.repeat(cells, o, axis=0), o, axis=1))
    assert len(np.unique(cells)) == cells.size
    assert not np.array_equal(W.config4_shifts(cfg, 2), sv)


def test_initial_state_is_separable_outer_product():
    cfg = W.CONFIG3.scaled((3, 2, 4, 2))
    rng = np.random.default_rng(0)
    coords = [np.sort(rng.uniform(lo, hi, n)) for lo, hi, n in zip(cfg.lo, cfg.hi, cfg.N)]
    gx, gv = W.initial_factors(cfg, coords)
    f = W.initial_state(cfg, coords)
    assert gx.shape == (cfg.X,) and gv.shape == (cfg.V,) and f.shape == (cfg.ndof,)
    # canonical layout: x_1 fastest
    F = f.reshape(cfg.N[3], cfg.N[2], cfg.N[1], cfg.N[0])
    p = (1, 3, 2, 4)     # (v2, v1, x2, x1)
    val = (1 + cfg.eps * (np.cos(cfg.k * coords[0][p[3]]) + np.cos(cfg.k * coords[1][p[2]]))) \
        * np.exp(-0.5 * (coords[2][p[1]] ** 2 + coords[3][p[0]] ** 2)) / (2 * np.pi)
    assert abs(F[p] - val) < 1e-16
    assert W.initial_state(cfg, coords, np.float32).dtype == np.float32


def test_paper_twostream_state_eq2():
    # PAPER.md eq. (2): f_eq integrates to 1 over v (each bracket to 2 sqrt(2 pi)), peaks near +-v0
    cfg = W.PAPER_TWOSTREAM
    assert cfg.order == 4 and cfg.cells == (60,) * 4 and cfg.extra["v0"] == 2.4
    v = np.linspace(-12, 12, 4801)
    x = np.array([0.0])
    gx, gv = W.initial_factors(cfg, [x, x, v, v])
    dv = v[1] - v[0]
    assert abs(gv.sum() * dv * dv - 1.0) < 1e-9
    assert abs(gx[0] - (1 + 2e-3)) < 1e-15
    F = gv.reshape(v.size, v.size)
    i, j = np.unravel_index(np.argmax(F), F.shape)
    assert abs(abs(v[i]) - 2.4) < 0.02 and abs(abs(v[j]) - 2.4) < 0.02
    # value at (v1, v2) = (v0, v0): (1 + e^{-2 v0^2})^2 / (8 pi)
    k = np.argmin(np.abs(v - 2.4))
    assert abs(F[k, k] - (1 + np.exp(-2 * 2.4 ** 2)) ** 2 / (8 * np.pi)) < 1e-12
