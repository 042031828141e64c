"""-m gpu: the CUDA translation sweep (sldg_translate / sldg_advect) against the CPU oracle,
element by element, on seeded inputs spanning several tiles and ragged tails."""
import numpy as np
import pytest

from paper_1907_08316_b200 import workloads as W
from tests.gpu_util import NPDT, TOL, dep_of, make_solver, rel_err

pytestmark = pytest.mark.gpu


def _random_shifts(rng, count, kind):
    if kind == "small":                    # |sigma| << 1 as in the physics v-sweeps
        return rng.uniform(-0.3, 0.3, count)
    if kind == "wide":                     # config-4 like
        return rng.uniform(-3.5, 3.5, count)
    if kind == "integer":                  # exact translation (P4)
        return rng.integers(-5, 6, count).astype(np.float64)
    if kind == "huge":                     # many wraps
        return rng.uniform(-1000.0, 1000.0, count)
    raise ValueError(kind)


def _sweep_case(oracle, cfg, dtype, dim, kind, seed):
    rng = np.random.default_rng(seed)
    s = make_solver(cfg, dtype)
    f0 = rng.uniform(0.0, 1.0, cfg.ndof).astype(NPDT[dtype])
    count = cfg.N[cfg.dx + dim] if dim < cfg.dx else cfg.X
    sigma = _random_shifts(rng, count, kind)
    s.set_initial(f0)
    s.translate(dim, sigma)
    got = s.get_f()
    ref = oracle.translate(f0.copy(), cfg.N, cfg.order, dim, sigma, dep_of(cfg.dx, dim))
    s.close()
    return got, ref


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("o", [1, 2, 3, 4, 5, 6])
@pytest.mark.parametrize("kind", ["small", "wide", "integer", "huge"])
def test_sweep_1p1(oracle, o, dtype, kind):
    cfg = W.Config("t11", 1, 1, (37, 29), o, (0.0, -3.0), (5.0, 3.0))
    for dim in (0, 1):
        got, ref = _sweep_case(oracle, cfg, dtype, dim, kind, 10 * o + dim)
        if kind == "integer":
            assert np.array_equal(got, ref)
        assert rel_err(got, ref) <= TOL[dtype]


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("o", [2, 3])
def test_sweep_2p2_every_direction(oracle, o, dtype):
    cfg = W.Config("t22", 2, 2, (12, 7, 9, 10), o, (0.0,) * 4, (12.0, 7.0, 9.0, 10.0))
    for dim in range(4):
        for kind in ("small", "wide"):
            got, ref = _sweep_case(oracle, cfg, dtype, dim, kind, 100 + dim)
            assert rel_err(got, ref) <= TOL[dtype], (dim, kind)


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("o", [2, 3])
def test_sweep_3p3_every_direction(oracle, o, dtype):
    cfg = W.Config("t33", 3, 3, (5, 4, 3, 6, 3, 4), o, (0.0,) * 6, (5.0, 4.0, 3.0, 6.0, 3.0, 4.0))
    for dim in range(6):
        got, ref = _sweep_case(oracle, cfg, dtype, dim, "wide", 200 + dim)
        assert rel_err(got, ref) <= TOL[dtype], dim


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_config4_reduced_twin_all_sweeps(oracle, dtype):
    """Config 4 recipe (uniform f from the counter generator, per-cell shifts) with every n_d
    divided by 8 and the full schedule of BASELINE.json configs[3]: 50 sweeps per direction
    (200 in all), element-wise parity after each direction."""
    cfg = W.CONFIG4.scaled((16, 16, 8, 8))
    s = make_solver(cfg, dtype)
    s.fill_uniform(W.SEED, W.TAG_F)
    f_host = W.uniform(W.SEED, W.TAG_F, np.arange(cfg.ndof, dtype=np.uint64)).astype(NPDT[dtype])
    assert np.array_equal(s.get_f(), f_host)        # device generator == host generator, bit for bit
    ref = f_host.copy()
    for dim in range(4):
        sigma = W.config4_shifts(cfg, dim)
        for _ in range(cfg.extra["sweeps_per_direction"]):
            s.translate(dim, sigma)
            oracle.translate(ref, cfg.N, cfg.order, dim, sigma, dep_of(cfg.dx, dim))
        assert rel_err(s.get_f(), ref) <= TOL[dtype], dim
    s.close()


def test_long_line_and_segments(oracle):
    """1+1 D with few long lines: the strided kernel splits lines into segments."""
    cfg = W.Config("long", 1, 1, (6, 300), 3, (0.0, -1.0), (1.0, 1.0))
    for kind in ("small", "wide", "huge"):
        got, ref = _sweep_case(oracle, cfg, "f64", 1, kind, 7)
        assert rel_err(got, ref) <= TOL["f64"], kind
    cfg = W.Config("long2", 2, 2, (4, 150, 3, 2), 2, (0.0,) * 4, (1.0,) * 4)
    got, ref = _sweep_case(oracle, cfg, "f64", 1, "wide", 8)
    assert rel_err(got, ref) <= TOL["f64"]


def test_single_cell_dimension(oracle):
    """Degenerate: one cell along the swept dimension (i* and i*+1 are the same cell)."""
    cfg = W.Config("one", 1, 1, (1, 5), 3, (0.0, -1.0), (1.0, 1.0))
    got, ref = _sweep_case(oracle, cfg, "f64", 0, "wide", 3)
    assert rel_err(got, ref) <= TOL["f64"]
    cfg = W.Config("one", 1, 1, (5, 1), 2, (0.0, -1.0), (1.0, 1.0))
    got, ref = _sweep_case(oracle, cfg, "f64", 1, "wide", 4)
    assert rel_err(got, ref) <= TOL["f64"]


def test_bad_arguments_fail_loudly():
    from paper_1907_08316_b200.sldg import SldgError
    cfg = W.Config("t", 1, 1, (4, 4), 2, (0.0, 0.0), (1.0, 1.0))
    s = make_solver(cfg, "f64")
    with pytest.raises(SldgError):
        s.translate(0, np.zeros(3))             # wrong count
    with pytest.raises(SldgError):
        s.advect(1, 0.1)                        # no E stored
    with pytest.raises(SldgError):
        s.poisson_E()                           # no rho
    s.close()
    with pytest.raises(SldgError):
        make_solver(W.Config("t", 1, 1, (4, 4), 7, (0.0, 0.0), (1.0, 1.0)), "f64")


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_plain_kernels_without_tma(oracle, dtype, monkeypatch):
    """SLDG_NO_TMA=1 selects the register-window / thread-per-cell kernels that also serve as
    fallbacks when the TMA preconditions fail; they must give the same results."""
    monkeypatch.setenv("SLDG_NO_TMA", "1")
    cfg = W.Config("t22", 2, 2, (12, 8, 9, 10), 3, (0.0,) * 4, (12.0, 8.0, 9.0, 10.0))
    for dim in range(4):
        got, ref = _sweep_case(oracle, cfg, dtype, dim, "wide", 300 + dim)
        assert rel_err(got, ref) <= TOL[dtype], dim
    cfg = W.Config("t11", 1, 1, (37, 29), 2, (0.0, -3.0), (5.0, 3.0))
    for dim in (0, 1):
        got, ref = _sweep_case(oracle, cfg, dtype, dim, "huge", 310 + dim)
        assert rel_err(got, ref) <= TOL[dtype], dim


def test_tma_and_plain_kernels_agree_bit_for_bit(monkeypatch):
    """Same FMA chains on both routes (D:O7): identical bits, at a size spanning many tiles."""
    cfg = W.CONFIG4.scaled((32, 16, 8, 8))
    outs = []
    for flag in ("0", "1"):
        monkeypatch.setenv("SLDG_NO_TMA", flag)
        s = make_solver(cfg, "f64")
        s.fill_uniform(W.SEED, W.TAG_F)
        for dim in range(4):
            s.translate(dim, W.config4_shifts(cfg, dim))
        outs.append(s.get_f())
        s.close()
    assert np.array_equal(outs[0], outs[1])


# ---------------------------------------------------------------- fused pairs (S:8(f) NEXT-1)

@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("amp", [3.5, 0.9])
@pytest.mark.parametrize("o", [1, 2, 3, 4])
@pytest.mark.parametrize("route", ["0", "1"])
def test_fused_pair_is_bitwise_the_two_sweeps_2p2(oracle, monkeypatch, o, amp, dtype, route):
    """amp = 0.9: |shift| < 1 cell, the regime of the fused v-kernels; amp = 3.5: a raw v-pair with wider shifts
    stays one (asynchronous) kernel whose blocks take the global-read fallback, or, with SLDG_ROUTE_WIDE=1, is
    routed to two single sweeps after a flag read-back (sldg.h); an x-pair is one kernel whatever the shift."""
    import torch
    monkeypatch.setenv("SLDG_ROUTE_WIDE", route)
    cfg = W.Config("p22", 2, 2, (11, 7, 9, 6), o, (0.0,) * 4, (11.0, 7.0, 9.0, 6.0))
    rng = np.random.default_rng(77 + o)
    f0 = rng.uniform(0.0, 1.0, cfg.ndof).astype(NPDT[dtype])
    for (k1, k2) in ((0, 1), (2, 3)):
        sig = []
        for k in (k1, k2):
            cnt = cfg.N[cfg.dx + k] if k < cfg.dx else cfg.X
            sig.append(rng.uniform(-amp, amp, cnt))
        a = make_solver(cfg, dtype)
        a.set_initial(f0)
        l0 = a.launch_count()
        a.translate_pair(k1, torch.from_numpy(sig[0]).cuda(), k2, torch.from_numpy(sig[1]).cuda())
        assert a.launch_count() - l0 == (4 if (k1 >= 2 and amp > 1.0 and route == "1") else 3)   # 2 table kernels + 1 or 2 sweeps
        fused = a.get_f()
        a.close()
        b = make_solver(cfg, dtype)
        b.set_initial(f0)
        b.translate(k1, sig[0])
        b.translate(k2, sig[1])
        seq = b.get_f()
        b.close()
        assert np.array_equal(fused, seq), (k1, k2)
        ref = f0.copy()
        oracle.translate(ref, cfg.N, cfg.order, k1, sig[0], dep_of(cfg.dx, k1))
        oracle.translate(ref, cfg.N, cfg.order, k2, sig[1], dep_of(cfg.dx, k2))
        assert rel_err(fused, ref) <= TOL[dtype], (k1, k2)


def test_fused_pairs_3p3_all_legal_pairs(oracle):
    import torch
    cfg = W.Config("p33", 3, 3, (5, 4, 3, 4, 3, 5), 2, (0.0,) * 6, (5.0, 4.0, 3.0, 4.0, 3.0, 5.0))
    rng = np.random.default_rng(5)
    f0 = rng.uniform(0.0, 1.0, cfg.ndof)
    for (k1, k2) in ((0, 1), (0, 2), (1, 2), (3, 4), (3, 5), (4, 5)):
        sig = [rng.uniform(-2.5, 2.5, cfg.N[cfg.dx + k] if k < cfg.dx else cfg.X) for k in (k1, k2)]
        s = make_solver(cfg, "f64")
        s.set_initial(f0)
        s.translate_pair(k1, torch.from_numpy(sig[0]).cuda(), k2, torch.from_numpy(sig[1]).cuda())
        fused = s.get_f()
        s.close()
        ref = f0.copy()
        oracle.translate(ref, cfg.N, cfg.order, k1, sig[0], dep_of(cfg.dx, k1))
        oracle.translate(ref, cfg.N, cfg.order, k2, sig[1], dep_of(cfg.dx, k2))
        assert rel_err(fused, ref) <= TOL["f64"], (k1, k2)


def test_fused_pair_rejects_mixed_groups():
    import torch
    from paper_1907_08316_b200.sldg import SldgError
    cfg = W.Config("p22", 2, 2, (4, 4, 4, 4), 2, (0.0,) * 4, (1.0,) * 4)
    s = make_solver(cfg, "f64")
    z = torch.zeros(cfg.N[3], dtype=torch.float64, device="cuda")
    zx = torch.zeros(cfg.X, dtype=torch.float64, device="cuda")
    with pytest.raises(SldgError):
        s.translate_pair(1, z, 2, zx)          # x_2 with v_1: the v-shift depends on the x_2 node
    with pytest.raises(SldgError):
        s.translate_pair(1, z, 0, z)           # not ascending
    s.close()


def test_step_fused_equals_step_unfused_bitwise(monkeypatch):
    cfg = W.CONFIG3.scaled((10, 8, 12, 6))
    outs = []
    # sweep fusion is bitwise neutral; rho accumulated in the x-sweep sums in another (fixed) grouping, so that
    # variant (the default) is compared at rounding level
    for flag, norho in (("0", "1"), ("1", "1"), ("0", "0")):
        monkeypatch.setenv("SLDG_NO_FUSE", flag)
        monkeypatch.setenv("SLDG_NO_FUSE_RHO", norho)
        s = make_solver(cfg, "f64")
        coords = [s.node_coords(d) for d in range(4)]
        s.set_initial(W.initial_state(cfg, coords))
        l0 = s.launch_count()
        for _ in range(3):
            s.step(cfg.dt)
        outs.append((s.get_f(), s.launch_count() - l0))
        s.close()
    assert np.array_equal(outs[0][0], outs[1][0])
    assert outs[0][1] < outs[1][1]             # the fused step really launches fewer sweeps
    assert rel_err(outs[2][0], outs[0][0]) <= 1e-13
    assert outs[2][1] < outs[0][1]             # ... and with rho inside the x-sweep one kernel fewer per step


@pytest.mark.parametrize("o", [1, 2, 3, 4, 5, 6])
def test_ab_tables_are_rounded_once(oracle, o):
    """Unit impulses pick out single entries of A(theta) and B(theta): the library's table
    (binary128 coefficients + double-double Horner) against the oracle's (long-double quadrature),
    both meant to be the exact value rounded once (D:O7) -- they may differ by one ulp at most."""
    n, nv = 5, 40
    cfg = W.Config("ab", 1, 1, (n, nv), o, (0.0, 0.0), (1.0, 1.0))
    rng = np.random.default_rng(o)
    theta = rng.uniform(0.0, 1.0, cfg.N[1])
    theta[:3] = (0.0, 0.5, 1.0 - 2.0 ** -40)
    f0 = np.zeros((cfg.N[1], cfg.N[0]))
    for q in range(cfg.N[1]):
        f0[q, 2 * o + (q % o)] = 1.0                  # impulse in cell 2, local node q % o
    f0 = f0.reshape(-1)
    s = make_solver(cfg, "f64")
    s.set_initial(f0)
    s.translate(0, -theta)                            # sigma = -theta  ->  m = 0, theta as given
    got = s.get_f()
    s.close()
    ref = oracle.translate(f0.copy(), cfg.N, o, 0, -theta, [1])
    nz = ref != 0.0
    assert np.array_equal(got == 0.0, ref == 0.0)
    # at most one ulp of the entry; entries that are tiny by cancellation (A near theta = 1, B near 0)
    # carry the oracle's long-double ABSOLUTE error of a few 1e-19 of the O(1) terms they are summed from
    assert np.all(np.abs(got - ref)[nz] <= np.spacing(np.abs(ref[nz])) + 2e-18)
    assert np.mean(got[nz] != ref[nz]) < 0.05                                   # and almost always the same double


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("amp", [2.5, 0.9])
@pytest.mark.parametrize("o", [1, 2, 3])
@pytest.mark.parametrize("one", ["0", "1"])
def test_fused_triple_is_bitwise_the_three_sweeps_3p3(oracle, monkeypatch, o, amp, dtype, one):
    """x_1,x_2,x_3 and v_1,v_2,v_3 in one pass each (o <= 2: the triple kernel; o = 3: pair + single);
    amp = 2.5: the raw v-triple with shifts of a cell or more takes the fused kernel's per-block fallback
    (one = "0") or, with SLDG_ROUTE_WIDE=1 (one = "1"), runs as single sweeps (sldg.h)."""
    import torch
    monkeypatch.setenv("SLDG_XTRIPLE_ONE", one)           # part-plane x-triple: one / two x_2-cells per thread
    monkeypatch.setenv("SLDG_ROUTE_WIDE", one)            # both settings of the wide-shift routing ride along
    cfg = W.Config("t33", 3, 3, (5, 4, 6, 4, 5, 3), o, (0.0,) * 6, (5.0, 4.0, 6.0, 4.0, 5.0, 3.0))
    rng = np.random.default_rng(31 + o)
    f0 = rng.uniform(0.0, 1.0, cfg.ndof).astype(NPDT[dtype])
    for ks in ((0, 1, 2), (3, 4, 5)):
        sig = [rng.uniform(-amp, amp, cfg.N[cfg.dx + k] if k < cfg.dx else cfg.X) for k in ks]
        a = make_solver(cfg, dtype)
        a.set_initial(f0)
        a.translate_triple(ks[0], torch.from_numpy(sig[0]).cuda(), ks[1], torch.from_numpy(sig[1]).cuda(),
                           ks[2], torch.from_numpy(sig[2]).cuda())
        fused = a.get_f()
        a.close()
        b = make_solver(cfg, dtype)
        b.set_initial(f0)
        for k, s_ in zip(ks, sig):
            b.translate(k, s_)
        seq = b.get_f()
        b.close()
        assert np.array_equal(fused, seq), ks
        ref = f0.copy()
        for k, s_ in zip(ks, sig):
            oracle.translate(ref, cfg.N, cfg.order, k, s_, dep_of(cfg.dx, k))
        assert rel_err(fused, ref) <= TOL[dtype], ks


def test_step_3p3_fused_equals_unfused_bitwise(monkeypatch):
    cfg = W.CONFIG5.scaled((6, 5, 4, 6, 4, 5))
    outs = []
    # sweep fusion is bitwise neutral; rho accumulated in the x-sweep sums in another (fixed) grouping, so that
    # variant (the default) is compared at rounding level
    for flag, norho in (("0", "1"), ("1", "1"), ("0", "0")):
        monkeypatch.setenv("SLDG_NO_FUSE", flag)
        monkeypatch.setenv("SLDG_NO_FUSE_RHO", norho)
        s = make_solver(cfg, "f64")
        coords = [s.node_coords(d) for d in range(6)]
        s.set_initial(W.initial_state(cfg, coords))
        l0 = s.launch_count()
        for _ in range(2):
            s.step(cfg.dt)
        outs.append((s.get_f(), s.launch_count() - l0))
        s.close()
    assert np.array_equal(outs[0][0], outs[1][0])
    assert outs[0][1] < outs[1][1]


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_no_write_outside_the_f_buffers(dtype):
    """Guard bands around caller-owned buffers (compute-sanitizer is closed on this pool): every
    kernel family on ragged sizes (tiles, chunks and segments that do not divide evenly) must leave
    the sentinels on both sides of both buffers untouched."""
    import torch
    from paper_1907_08316_b200.sldg import Sldg
    G = 4096
    tdt = torch.float64 if dtype == "f64" else torch.float32
    for dx, dv, cells, o in ((2, 2, (11, 7, 9, 5), 3), (3, 3, (5, 3, 4, 3, 5, 3), 2), (1, 1, (37, 29), 4),
                             (2, 2, (10, 6, 7, 5), 2)):
        cfg = W.Config("g", dx, dv, cells, o, (0.0,) * (dx + dv), tuple(float(c) for c in cells), dt=0.1)
        n = cfg.ndof
        big = [torch.full((n + 2 * G,), -777.0, dtype=tdt, device="cuda") for _ in range(2)]
        bufs = [b[G:G + n] for b in big]
        s = Sldg(cfg.dx, cfg.dv, cfg.cells, cfg.order, cfg.lo, cfg.hi, dtype=dtype, buffers=bufs)
        s.fill_uniform(W.SEED, 0)
        rng = np.random.default_rng(1)
        D = dx + dv
        sig = [torch.from_numpy(rng.uniform(-3.5, 3.5, cfg.N[dx + k] if k < dx else cfg.X)).cuda() for k in range(D)]
        for k in range(D):
            s.translate(k, sig[k])
        s.translate_pair(0, sig[0], 1, sig[1]) if dx >= 2 else None
        s.translate_pair(dx, sig[dx], dx + 1, sig[dx + 1]) if dv >= 2 else None
        if dx == 3:
            s.translate_triple(0, sig[0], 1, sig[1], 2, sig[2])
            s.translate_triple(3, sig[3], 4, sig[4], 5, sig[5])
        s.step(0.1)
        s.diagnostics()
        s.moments()
        torch.cuda.synchronize()
        for b in big:
            assert bool((b[:G] == -777.0).all()) and bool((b[G + n:] == -777.0).all()), (cells, o)
        assert bool(torch.isfinite(s.current()).all())
        s.close()


def test_create_destroy_does_not_leak_device_memory():
    import torch
    cfg = W.Config("leak", 2, 2, (8, 8, 8, 8), 3, (0.0,) * 4, (1.0,) * 4, dt=0.1)
    def cycle():
        s = make_solver(cfg, "f64")
        s.fill_uniform(1, 0)
        s.step(0.1); s.step(0.1); s.step(0.1)        # includes a captured graph
        s.diagnostics(); s.moments()
        s.close()
    cycle()
    torch.cuda.synchronize(); torch.cuda.empty_cache()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(40):
        cycle()
    torch.cuda.synchronize(); torch.cuda.empty_cache()
    free1, _ = torch.cuda.mem_get_info()
    assert free0 - free1 < 8 * 1024 * 1024, (free0, free1)


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("o", [1, 2, 3, 4])
@pytest.mark.parametrize("kind", ["small-mixed-sign", "small-one-sign", "some-large"])
def test_tile_staged_v_pair(oracle, o, dtype, kind, monkeypatch):
    """The TMA-tile staged v-pair (both k1-neighbours staged; lanes may look left or right, early or
    late, independently) and its per-block fallback for offsets outside {0, n-1}: bitwise equal to the
    two single sweeps and within tolerance of the oracle."""
    import torch
    monkeypatch.setenv("SLDG_TILE_PAIR", "1")              # also at o <= 2
    cfg = W.Config("tile", 2, 2, (16, 4, 8, 5), o, (0.0,) * 4, (16.0, 4.0, 8.0, 5.0))
    assert cfg.X % 32 == 0
    rng = np.random.default_rng(1000 + o)
    f0 = rng.uniform(0.0, 1.0, cfg.ndof).astype(NPDT[dtype])
    x = np.arange(cfg.X)
    if kind == "small-mixed-sign":
        sig = [0.4 * np.sin(2 * np.pi * x / 23.0), 0.7 * np.cos(2 * np.pi * x / 41.0)]
    elif kind == "small-one-sign":
        sig = [0.2 + 0.1 * np.sin(x), -0.5 + 0.3 * np.cos(x)]
    else:
        sig = [0.4 * np.sin(2 * np.pi * x / 23.0), 0.7 * np.cos(2 * np.pi * x / 41.0)]
        sig[0][40:44] = 2.3                                  # one tile with offsets outside {0, n-1}
        sig[1][cfg.X - 7] = -1.7
    a = make_solver(cfg, dtype)
    a.set_initial(f0)
    b = make_solver(cfg, dtype)
    b.set_initial(f0)
    ref = f0.copy()
    if kind == "some-large":
        # the raw call would route shifts of a cell or more to single sweeps (sldg.h); the physics call does not
        # check, so it reaches the kernel's per-block fallback: sigma = -E dt / h_v with dt = 1
        g = oracle.Grid(cfg.dx, cfg.dv, cfg.cells, cfg.order, cfg.lo, cfg.hi)
        E = np.stack([-sig[a_] * (cfg.hi[2 + a_] - cfg.lo[2 + a_]) / cfg.cells[2 + a_] for a_ in range(2)])
        a.set_E(E); b.set_E(E)
        a.advect_pair(2, 3, 1.0)
        b.advect(2, 1.0); b.advect(3, 1.0)
        g.advect(ref, 2, 1.0, E); g.advect(ref, 3, 1.0, E)
    else:
        a.translate_pair(2, torch.from_numpy(sig[0]).cuda(), 3, torch.from_numpy(sig[1]).cuda())
        b.translate(2, sig[0])
        b.translate(3, sig[1])
        oracle.translate(ref, cfg.N, cfg.order, 2, sig[0], [0, 1])
        oracle.translate(ref, cfg.N, cfg.order, 3, sig[1], [0, 1])
    fused = a.get_f()
    seq = b.get_f()
    a.close(); b.close()
    assert np.array_equal(fused, seq)
    assert rel_err(fused, ref) <= TOL[dtype]


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("o", [1, 2])
@pytest.mark.parametrize("kind", ["small-mixed-sign", "small-one-sign", "some-large"])
def test_tile_staged_v_triple(oracle, o, dtype, kind):
    """The TMA-tile staged v-triple (both neighbours staged in v_1 and v_2, early/late in v_3) and its
    per-block fallback: bitwise equal to the three single sweeps, within tolerance of the oracle."""
    import torch
    cfg = W.Config("tile3", 3, 3, (4, 4, 2, 4, 8, 5), o, (0.0,) * 6, (4.0, 4.0, 2.0, 4.0, 8.0, 5.0))
    assert cfg.X % 32 == 0
    rng = np.random.default_rng(2000 + o)
    f0 = rng.uniform(0.0, 1.0, cfg.ndof).astype(NPDT[dtype])
    x = np.arange(cfg.X)
    if kind == "small-one-sign":
        sig = [0.2 + 0.1 * np.sin(x), -0.5 + 0.3 * np.cos(x), 0.6 + 0.2 * np.sin(0.3 * x)]
    else:
        sig = [0.4 * np.sin(2 * np.pi * x / 23.0), 0.7 * np.cos(2 * np.pi * x / 41.0), 0.9 * np.sin(2 * np.pi * x / 17.0)]
        if kind == "some-large":
            sig[0][3:6] = 2.3
            sig[2][cfg.X - 7] = -1.7
    a = make_solver(cfg, dtype)
    a.set_initial(f0)
    b = make_solver(cfg, dtype)
    b.set_initial(f0)
    ref = f0.copy()
    if kind == "some-large":
        # physics call (no routing of wide shifts): reaches the kernel's per-block fallback
        g = oracle.Grid(cfg.dx, cfg.dv, cfg.cells, cfg.order, cfg.lo, cfg.hi)
        E = np.stack([-sig[a_] * (cfg.hi[3 + a_] - cfg.lo[3 + a_]) / cfg.cells[3 + a_] for a_ in range(3)])
        a.set_E(E); b.set_E(E)
        a.advect_triple(3, 4, 5, 1.0)
        for k in (3, 4, 5):
            b.advect(k, 1.0)
            g.advect(ref, k, 1.0, E)
    else:
        a.translate_triple(3, torch.from_numpy(sig[0]).cuda(), 4, torch.from_numpy(sig[1]).cuda(),
                           5, torch.from_numpy(sig[2]).cuda())
        for k, s_ in zip((3, 4, 5), sig):
            b.translate(k, s_)
            oracle.translate(ref, cfg.N, cfg.order, k, s_, [0, 1, 2])
    fused = a.get_f()
    seq = b.get_f()
    a.close(); b.close()
    assert np.array_equal(fused, seq)
    assert rel_err(fused, ref) <= TOL[dtype]


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("o", [2, 3, 4])
def test_two_live_contexts_of_different_size_interleaved(o, dtype):
    """The dynamic shared-memory opt-in belongs to (device, kernel), not to a context, and setting it stores the
    exact value: a second, smaller context that uses the same kernels must not lower what the first one's launches
    need.  Two live contexts of the same dtype and order, a large and a small grid, take turns through
    single sweeps, fused pairs and Strang steps; the large one must come out bit for bit as when it runs alone."""
    import torch
    big = W.Config("big", 2, 2, (40, 36, 24, 20), o, (0.0, 0.0, -4.0, -4.0), (4 * np.pi, 4 * np.pi, 4.0, 4.0))
    small = W.Config("small", 2, 2, (5, 4, 4, 3), o, (0.0, 0.0, -4.0, -4.0), (4 * np.pi, 4 * np.pi, 4.0, 4.0))
    rng = np.random.default_rng(77)
    fb = rng.uniform(0.0, 1.0, big.ndof).astype(NPDT[dtype])
    fs = rng.uniform(0.0, 1.0, small.ndof).astype(NPDT[dtype])

    def shifts(cfg, seed):
        r = np.random.default_rng(seed)
        return [r.uniform(-0.4, 0.4, cfg.N[cfg.dx + d] if d < cfg.dx else cfg.X) for d in range(4)]

    def work(s, cfg, seed):
        sig = shifts(cfg, seed)
        for d in range(4):
            s.translate(d, sig[d])
        dev = [torch.from_numpy(x).cuda() for x in sig]
        s.translate_pair(0, dev[0], 1, dev[1])
        s.translate_pair(2, dev[2], 3, dev[3])
        s.step(0.05)

    alone = make_solver(big, dtype)
    alone.set_initial(fb)
    work(alone, big, 1)
    work(alone, big, 2)
    want = alone.get_f()
    alone.close()

    a, b = make_solver(big, dtype), make_solver(small, dtype)
    a.set_initial(fb)
    b.set_initial(fs)
    work(a, big, 1)
    work(b, small, 3)          # same kernels, smaller shared-memory requests
    work(a, big, 2)            # failed with "invalid value" when the opt-in was remembered per context
    work(b, small, 4)
    got = a.get_f()
    a.close(); b.close()
    assert np.all(np.isfinite(got))
    assert np.array_equal(got, want)


def test_wide_shift_seen_marks_fused_v_sweeps_outside_their_regime():
    """sldg_wide_shift_seen: the fused v-sweeps never check |E| dt < h_v (they fall back per block, same bits, slower);
    the table assembly leaves a sticky mark instead, so the cost is not silent.  x-groups and single sweeps, which
    take any shift in their stride, never raise it."""
    import torch
    cfg = W.Config("wide", 2, 2, (8, 6, 8, 8), 3, (0.0, 0.0, -4.0, -4.0), (4 * np.pi, 4 * np.pi, 4.0, 4.0))
    hv = 1.0                                              # (4 - -4) / 8
    rng = np.random.default_rng(9)
    s = make_solver(cfg, "f64")
    s.set_initial(rng.uniform(0.0, 1.0, cfg.ndof))
    assert s.wide_shift_seen() is False
    wide_v = torch.from_numpy(rng.uniform(-3.5, 3.5, cfg.N[2])).cuda()
    wide_w = torch.from_numpy(rng.uniform(-3.5, 3.5, cfg.N[3])).cuda()
    s.translate_pair(0, wide_v, 1, wide_w)                # x-pair: any shift is its home ground
    s.translate(2, rng.uniform(-3.5, 3.5, cfg.X))         # single v-sweep: likewise
    s.set_E(0.3 * hv * np.sin(np.arange(2 * cfg.X)).reshape(2, cfg.X))
    s.advect_pair(2, 3, 1.0)                              # |E| dt < h_v: the regime the fused v-pair is built for
    s.step(0.05)
    assert s.wide_shift_seen() is False
    s.set_E(2.5 * hv * np.sin(np.arange(2 * cfg.X)).reshape(2, cfg.X))
    s.advect_pair(2, 3, 1.0)                              # some lines move by more than a cell
    assert s.wide_shift_seen(reset=True) is True
    assert s.wide_shift_seen() is False                   # the reset took
    small_x = torch.from_numpy(rng.uniform(-0.4, 0.4, cfg.X)).cuda()
    wide_x = torch.from_numpy(rng.uniform(-2.5, 2.5, cfg.X)).cuda()
    s.translate_pair(2, small_x, 3, small_x)
    assert s.wide_shift_seen() is False
    s.translate_pair(2, small_x, 3, wide_x)               # raw fused v-call, second table wide
    assert s.wide_shift_seen() is True
    s.close()
