"""-m gpu: the launch configurations bench.py times (BASELINE.json configs 3, 4, 5 at FULL size).

The oracle cannot sweep 43 GB in seconds, so parity is checked on sampled outputs it can compute one
by one: after a sweep, seeded random lines are pulled from the pre- and
post-sweep device buffers and compared with the oracle's 1-D rule on the same line and shift (a
D-dimensional sweep IS the 1-D rule on every line: P:69, oracle pin P12); plus properties that hold
at any size: mass conservation (P5) and L2 non-increase (P8) per sweep."""
import numpy as np
import pytest

from paper_1907_08316_b200 import workloads as W
from tests.gpu_util import NPDT, TOL, make_solver

pytestmark = pytest.mark.gpu

NLINES = 1500


def _need_gb(gb):
    import torch
    free, _ = torch.cuda.mem_get_info()
    if free < gb * 1e9:
        pytest.skip("needs %.0f GB of device memory" % gb)


def _sampled_line_parity(oracle, s, cfg, dtype, dim, sigma, rng):
    import torch
    D = cfg.dx + cfg.dv
    N = cfg.N
    inner = int(np.prod(N[:dim])) if dim else 1
    outer = int(np.prod(N[dim + 1:])) if dim + 1 < D else 1
    Nk = N[dim]
    pre = s.current()
    s.translate(dim, sigma)
    post = s.current()
    assert pre.data_ptr() != post.data_ptr()
    oo = rng.integers(0, outer, NLINES)
    ii = rng.integers(0, inner, NLINES)
    # always include the corners (first/last line of the array: tile and tail handling)
    oo[:2] = (0, outer - 1)
    ii[:2] = (0, inner - 1)
    base = torch.from_numpy(oo * Nk * inner + ii).cuda()
    idx = base[:, None] + torch.arange(Nk, device="cuda")[None, :] * inner
    u_old = pre[idx].cpu().numpy()
    u_new = post[idx].cpu().numpy()
    if dim < cfg.dx:
        qdiv = int(np.prod(N[dim + 1: cfg.dx + dim]))
        q = (oo // qdiv) % N[cfg.dx + dim]
    else:
        q = ii % cfg.X
    sig = np.asarray(sigma.cpu().numpy() if hasattr(sigma, "cpu") else sigma)
    worst = 0.0
    cache = {}
    for r in range(NLINES):
        key = float(sig[q[r]])
        if key not in cache:
            m, th = oracle.shift_split(key)
            A, B = oracle.assemble_AB(cfg.order, th)
            cache[key] = (m, A.astype(NPDT[dtype]), B.astype(NPDT[dtype]))
        m, A, B = cache[key]
        ref = oracle.translate_line(cfg.order, A, B, m, u_old[r])
        worst = max(worst, float(np.max(np.abs(u_new[r].astype(np.float64) - ref))))
    return worst / float(np.max(np.abs(u_old)))


def _check_config(oracle, cfg, dtype, shifts_of, gb):
    import torch
    _need_gb(gb)
    rng = np.random.default_rng(42)
    s = make_solver(cfg, dtype)
    if cfg.kind == "uniform":
        s.fill_uniform(W.SEED, W.TAG_F)
        # the device generator against the host recipe on a sample of the 5.4e9 values
        g = rng.integers(0, cfg.ndof, 100000)
        g[:2] = (0, cfg.ndof - 1)
        dev = s.current()[torch.from_numpy(g).cuda()].cpu().numpy()
        assert np.array_equal(dev, W.uniform(W.SEED, W.TAG_F, g.astype(np.uint64)).astype(NPDT[dtype]))
    else:
        # separable analytic initial state built on the device from the library's node coordinates
        coords = [s.node_coords(d) for d in range(cfg.dx + cfg.dv)]
        gx, gv = W.initial_factors(cfg, coords)
        f0 = torch.outer(torch.from_numpy(gv).cuda(), torch.from_numpy(gx).cuda()).reshape(-1)
        s.set_initial(f0.to(s.tdtype).contiguous())
        del f0
    mass0, l20, _ = s.diagnostics()
    rel_mass = 1e-12 if dtype == "f64" else 1e-6
    for dim in range(cfg.dx + cfg.dv):
        sigma = torch.from_numpy(np.ascontiguousarray(shifts_of(dim))).cuda()
        err = _sampled_line_parity(oracle, s, cfg, dtype, dim, sigma, rng)
        assert err <= TOL[dtype], (cfg.name, dtype, dim, err)
        mass, l2, _ = s.diagnostics()
        assert abs(mass - mass0) <= rel_mass * abs(mass0), (dim, mass, mass0)      # P5
        assert l2 <= l20 * (1 + rel_mass), (dim, l2, l20)                           # P8
        l20 = l2
    s.close()
    torch.cuda.empty_cache()


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_config4_full_size_sampled_lines(oracle, dtype):
    cfg = W.CONFIG4
    _check_config(oracle, cfg, dtype, lambda dim: W.config4_shifts(cfg, dim), 95 if dtype == "f64" else 48)


def _physics_like_shifts(cfg):
    def shifts(dim):
        cnt = cfg.N[cfg.dx + dim] if dim < cfg.dx else cfg.X
        if dim < cfg.dx:      # sigma = v dt/2 / h_x at equispaced stand-ins for the v-nodes
            va = cfg.dx + dim
            h = (cfg.hi[dim] - cfg.lo[dim]) / cfg.cells[dim]
            return np.linspace(cfg.lo[va], cfg.hi[va], cnt) * 0.5 * cfg.dt / h
        return 0.04 * (W.uniform(W.SEED, W.TAG_SHIFT + dim, np.arange(cnt, dtype=np.uint64)) - 0.5)
    return shifts


def test_config3_full_size_sampled_lines(oracle):
    _check_config(oracle, W.CONFIG3, "f64", _physics_like_shifts(W.CONFIG3), 5)


def test_config5_full_size_sampled_lines(oracle):
    _check_config(oracle, W.CONFIG5, "f64", _physics_like_shifts(W.CONFIG5), 70)


def test_config3_full_size_one_step_against_full_oracle(oracle):
    """One full Strang step of config 3 (2.1 GB) against the complete oracle, element by element."""
    import torch
    _need_gb(5)
    cfg = W.CONFIG3
    g = oracle.Grid(cfg.dx, cfg.dv, cfg.cells, cfg.order, cfg.lo, cfg.hi)
    f = W.initial_state(cfg, [g.coords(d) for d in range(4)], np.float64)
    s = make_solver(cfg, "f64")
    s.set_initial(f)
    s.step(cfg.dt)
    g.step(f, cfg.dt)
    got = s.get_f()
    err = float(np.max(np.abs(got - f)) / np.max(np.abs(f)))
    m, l2, ee = s.diagnostics()
    mr, l2r, eer = g.diagnostics(f)
    s.close()
    torch.cuda.empty_cache()
    assert err <= TOL["f64"]
    assert abs(ee - eer) <= 1e-12 * eer and abs(m - mr) <= 1e-12 * mr and abs(l2 - l2r) <= 1e-12 * l2r


def _fused_vs_single_fullsize(cfg, dtype, groups, shifts_of, gb):
    """Fused pair / triple at full size against the same single sweeps, bit for bit (two solvers).
    The single sweeps are the ones checked against the oracle by the sampled-line tests above."""
    import torch
    _need_gb(gb)
    a = make_solver(cfg, dtype)
    b = make_solver(cfg, dtype)
    a.fill_uniform(W.SEED, W.TAG_F)
    b.fill_uniform(W.SEED, W.TAG_F)
    for ks in groups:
        sh = [torch.from_numpy(np.ascontiguousarray(shifts_of(k))).cuda() for k in ks]
        if len(ks) == 3:
            a.translate_triple(ks[0], sh[0], ks[1], sh[1], ks[2], sh[2])
        else:
            a.translate_pair(ks[0], sh[0], ks[1], sh[1])
        for k, s_ in zip(ks, sh):
            b.translate(k, s_)
        fa, fb = a.current(), b.current()
        same = True
        chunk = 1 << 28
        for i in range(0, fa.numel(), chunk):
            same = same and bool(torch.equal(fa[i:i + chunk], fb[i:i + chunk]))
        assert same, ks
    a.close()
    b.close()
    torch.cuda.empty_cache()


def _smooth_shifts(cfg):
    def shifts(dim):
        cnt = cfg.N[cfg.dx + dim] if dim < cfg.dx else cfg.X
        if dim < cfg.dx:
            va = cfg.dx + dim
            h = (cfg.hi[dim] - cfg.lo[dim]) / cfg.cells[dim]
            return np.linspace(cfg.lo[va], cfg.hi[va], cnt) * 0.5 * cfg.dt / h
        return 0.3 * np.sin(2 * np.pi * np.arange(cnt) / cfg.N[0] + 0.1 * dim)     # smooth in x like E
    return shifts


def test_config5_full_size_fused_triples_equal_single_sweeps():
    _fused_vs_single_fullsize(W.CONFIG5, "f64", [(0, 1, 2), (3, 4, 5)], _smooth_shifts(W.CONFIG5), 140)


def test_config4_fp32_full_size_fused_pairs_equal_single_sweeps():
    cfg = W.CONFIG4
    _fused_vs_single_fullsize(cfg, "f32", [(0, 1), (2, 3)], lambda d: W.config4_shifts(cfg, d), 95)


def test_config3_full_size_fused_pairs_equal_single_sweeps():
    _fused_vs_single_fullsize(W.CONFIG3, "f64", [(0, 1), (2, 3)], _smooth_shifts(W.CONFIG3), 10)
