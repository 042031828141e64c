"""Seeded, synthetic input generators for the BASELINE.json configs.

This module serves BOTH the CUDA library's tests/bench and the CPU oracle.  It
holds none of the method's arithmetic: no Gauss-Legendre rule, no A/B matrices,
no sweep, reduction or Poisson code.  Node coordinates are passed IN (from
whichever side is being driven); what comes out is plain data: grid arguments,
initial states evaluated at those coordinates, the counter-based uniform
generator U(seed, tag, g) and the config-4 shift tables.

The paper measures on no dataset: every workload is an analytic initial state
(eq. (2)) or, for the sweep microbenchmark, seeded
uniform noise (BASELINE.json configs[3]); DESIGN.md "Input recipe".
"""
from dataclasses import dataclass, field
from typing import Tuple

import numpy as np

SEED = 190708316  # the arXiv number, SURVEY.md section 8(d) config 4

# stream tags of U(seed, tag, g)
TAG_F = 0           # f[g], g = canonical linear index
TAG_SHIFT = 16      # + dim: one draw per cell of the dimension(s) the shift depends on


@dataclass(frozen=True)
class Config:
    """Arguments of sldg_create plus the run recipe of one BASELINE.json config."""
    name: str
    dx: int
    dv: int
    cells: Tuple[int, ...]
    order: int
    lo: Tuple[float, ...]
    hi: Tuple[float, ...]
    dt: float = 0.0
    steps: int = 0
    kind: str = "landau"     # landau | twostream | uniform
    eps: float = 0.0
    k: float = 0.0
    extra: dict = field(default_factory=dict)

    @property
    def N(self):
        return tuple(int(c) * self.order for c in self.cells)

    @property
    def X(self):
        return int(np.prod(self.N[: self.dx]))

    @property
    def V(self):
        return int(np.prod(self.N[self.dx:]))

    @property
    def ndof(self):
        return self.X * self.V

    def scaled(self, cells, name=None, steps=None):
        """Same physics/recipe on another cell count (the 'reduced twin' of DESIGN.md)."""
        c = tuple(int(x) for x in cells)
        hi = self.hi
        if self.kind == "uniform":          # unit cells: hi = n_d
            hi = tuple(float(x) for x in c)
        return Config(name or (self.name + "-twin"), self.dx, self.dv, c, self.order, self.lo, hi,
                      self.dt, self.steps if steps is None else steps, self.kind, self.eps, self.k,
                      dict(self.extra))


_PI = float(np.pi)

CONFIG1 = Config("config1-landau-1+1", 1, 1, (64, 64), 2, (0.0, -6.0), (4 * _PI, 6.0),
                 dt=0.1, steps=200, kind="landau", eps=0.01, k=0.5)
CONFIG2 = Config("config2-twostream-1+1", 1, 1, (256, 256), 3, (0.0, -9.0), (10 * _PI, 9.0),
                 dt=0.05, steps=400, kind="twostream", eps=0.001, k=0.2)
CONFIG3 = Config("config3-landau-2+2", 2, 2, (64, 64, 64, 64), 2, (0.0, 0.0, -6.0, -6.0),
                 (4 * _PI, 4 * _PI, 6.0, 6.0), dt=0.1, steps=20, kind="landau", eps=0.01, k=0.5)
CONFIG4 = Config("config4-sweep-2+2", 2, 2, (128, 128, 64, 64), 3, (0.0, 0.0, 0.0, 0.0),
                 (128.0, 128.0, 64.0, 64.0), kind="uniform", extra={"sweeps_per_direction": 50})
CONFIG5 = Config("config5-landau-3+3", 3, 3, (20,) * 6, 2, (0.0, 0.0, 0.0, -6.0, -6.0, -6.0),
                 (4 * _PI,) * 3 + (6.0,) * 3, dt=0.1, steps=5, kind="landau", eps=0.01, k=0.5)

# S:8(f) NEXT-2 -- the paper's validation run (section 8, eq. (2)): 2+2 D two-stream instability,
# 60^4 cells, o = 4, t <= 100.  The paper does not print its time step: dt = 0.1 is this build's choice.
PAPER_TWOSTREAM = Config("paper-twostream-2+2", 2, 2, (60, 60, 60, 60), 4, (0.0, 0.0, -6.0, -6.0),
                         (10 * _PI, 10 * _PI, 6.0, 6.0), dt=0.1, steps=1000, kind="twostream2",
                         eps=1e-3, k=0.2, extra={"v0": 2.4})

# S:8(f) NEXT-3 -- the mixed-dimension set-ups of the paper's section 7 (1+3 D and 2+3 D at o = 4; the
# paper's grid sizes are lost with its figures: these are this build's choices, ~1e9 and ~3.6e9 DOF).
MIXED13 = Config("mixed-landau-1+3", 1, 3, (32, 48, 48, 48), 4, (0.0, -6.0, -6.0, -6.0),
                 (4 * _PI, 6.0, 6.0, 6.0), dt=0.1, steps=5, kind="landau", eps=0.01, k=0.5)
MIXED23 = Config("mixed-landau-2+3", 2, 3, (16, 16, 24, 24, 24), 4, (0.0, 0.0, -6.0, -6.0, -6.0),
                 (4 * _PI, 4 * _PI, 6.0, 6.0, 6.0), dt=0.1, steps=3, kind="landau", eps=0.01, k=0.5)

CONFIGS = {c.name.split("-")[0]: c for c in (CONFIG1, CONFIG2, CONFIG3, CONFIG4, CONFIG5)}


# ---- analytic initial states, separable: f0[v][x] = gx[x] * gv[v] ---------------------------

def _flat_outer(parts):
    """prod_a parts[a][p_a] as a flat array, index 0 fastest (canonical order)."""
    out = np.asarray(parts[0], dtype=np.float64)
    for p in parts[1:]:
        out = np.multiply.outer(np.asarray(p, dtype=np.float64), out).reshape(-1)
    return np.ascontiguousarray(out)


def _flat_sum(parts):
    out = np.asarray(parts[0], dtype=np.float64)
    for p in parts[1:]:
        out = np.add.outer(np.asarray(p, dtype=np.float64), out).reshape(-1)
    return np.ascontiguousarray(out)


def initial_factors(cfg, coords):
    """(gx[X], gv[V]) in fp64 with f0 = outer(gv, gx); coords[d] = node coordinates of dim d."""
    assert len(coords) == cfg.dx + cfg.dv
    xs, vs = coords[: cfg.dx], coords[cfg.dx:]
    if cfg.kind == "landau":
        # (1 + eps sum_a cos(k x_a)) * exp(-|v|^2/2) / (2 pi)^{dv/2}
        gx = 1.0 + cfg.eps * _flat_sum([np.cos(cfg.k * np.asarray(x)) for x in xs])
        gv = _flat_outer([np.exp(-0.5 * np.asarray(v) ** 2) / np.sqrt(2.0 * np.pi) for v in vs])
    elif cfg.kind == "twostream":
        # (1 + eps cos(k x)) * v^2 exp(-v^2/2) / sqrt(2 pi)   (BASELINE.json configs[1])
        gx = 1.0 + cfg.eps * _flat_sum([np.cos(cfg.k * np.asarray(x)) for x in xs])
        gv = _flat_outer([np.asarray(v) ** 2 * np.exp(-0.5 * np.asarray(v) ** 2) / np.sqrt(2.0 * np.pi)
                          for v in vs])
    elif cfg.kind == "twostream2":
        # the paper's own validation state, eq. (2):
        # (1 + eps sum_a cos(k x_a)) * prod_a (exp(-(v_a-v0)^2/2) + exp(-(v_a+v0)^2/2)) / (2 sqrt(2 pi))
        # (= 1/(8 pi) times the two brackets for d_v = 2)
        v0 = float(cfg.extra["v0"])
        gx = 1.0 + cfg.eps * _flat_sum([np.cos(cfg.k * np.asarray(x)) for x in xs])
        gv = _flat_outer([(np.exp(-0.5 * (np.asarray(v) - v0) ** 2) + np.exp(-0.5 * (np.asarray(v) + v0) ** 2))
                          / (2.0 * np.sqrt(2.0 * np.pi)) for v in vs])
    else:
        raise ValueError("config kind %r has no analytic initial state" % cfg.kind)
    return gx, gv


def initial_state(cfg, coords, dtype=np.float64):
    """f0 flat in canonical layout, evaluated in fp64 then rounded to dtype."""
    if cfg.kind == "uniform":
        return uniform(SEED, TAG_F, np.arange(cfg.ndof, dtype=np.uint64)).astype(dtype)
    gx, gv = initial_factors(cfg, coords)
    return np.multiply.outer(gv, gx).reshape(-1).astype(dtype)


# ---- counter-based uniform generator ------------------------------------------------------

_M64 = np.uint64(0xFFFFFFFFFFFFFFFF)


def mix64(seed, tag, g):
    """Stateless 64-bit mixer (the splitmix64 finaliser) of the triple (seed, tag, g).

    x = g + 0x9E3779B97F4A7C15*(tag+1) + 0xD1B54A32D192ED03*seed   (mod 2^64), then
    x ^= x>>30; x *= 0xBF58476D1CE4E5B9; x ^= x>>27; x *= 0x94D049BB133111EB; x ^= x>>31.
    The CUDA library's fill kernel restates the same recipe (csrc/fill.cu).
    """
    g = np.asarray(g, dtype=np.uint64)
    with np.errstate(over="ignore"):
        off = (np.uint64(0x9E3779B97F4A7C15) * np.uint64(int(tag) + 1)
               + np.uint64(0xD1B54A32D192ED03) * np.uint64(int(seed)))
        x = g + off
        x = x ^ (x >> np.uint64(30))
        x = x * np.uint64(0xBF58476D1CE4E5B9)
        x = x ^ (x >> np.uint64(27))
        x = x * np.uint64(0x94D049BB133111EB)
        x = x ^ (x >> np.uint64(31))
    return x


def uniform(seed, tag, g):
    """U(seed, tag, g) in [0,1): top 53 bits of mix64 times 2^-53, fp64."""
    return (mix64(seed, tag, g) >> np.uint64(11)).astype(np.float64) * (2.0 ** -53)


def config4_shifts(cfg, dim, seed=SEED, amplitude=3.5):
    """Per-node shift table (cell widths) of a config-4 sweep along `dim` (R7).

    One draw sigma = -amplitude + 2*amplitude*U(seed, TAG_SHIFT+dim, c) per CELL c of the
    dimension(s) the shift depends on, replicated to that cell's nodes:
      dim = x_a : c = cell of v_a            -> table of N_{v_a} entries
      dim = v_a : c = (i_1, .., i_dx), i_1 fastest -> table of X entries (x_1 fastest)
    """
    o = cfg.order
    if dim < cfg.dx:
        n = cfg.cells[cfg.dx + dim]
        draw = -amplitude + 2.0 * amplitude * uniform(seed, TAG_SHIFT + dim, np.arange(n, dtype=np.uint64))
        return np.repeat(draw, o)
    ncell = int(np.prod(cfg.cells[: cfg.dx]))
    draw = -amplitude + 2.0 * amplitude * uniform(seed, TAG_SHIFT + dim, np.arange(ncell, dtype=np.uint64))
    draw = draw.reshape(tuple(reversed(cfg.cells[: cfg.dx])))      # C order: x_1 fastest
    for ax in range(cfg.dx):
        draw = np.repeat(draw, o, axis=ax)
    return np.ascontiguousarray(draw.reshape(-1))
