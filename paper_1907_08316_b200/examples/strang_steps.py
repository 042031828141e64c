"""Strang steps (sldg_step) of a named Vlasov-Poisson configuration on one B200, with the time
buckets of the paper's Fig. 5 ("advection x", "compute rho", "poisson",
"advection v").

    python -m paper_1907_08316_b200.examples.strang_steps --config config5 [--steps 5] [--warmup 2]
           [--dtype f64] [--order O] [--cells n1,n2,..] [--buckets] [--diagnostics] [--merged]

--config: config1 | config2 | config3 | config5 | mixed13 | mixed23 | twostream (the paper's eq. (2) run).
--buckets issues the same sequence as sldg_step through the public calls (advect pair/triple, compute_rho,
poisson_E) with CUDA events between the categories; without it the step is one sldg_step call.
--merged runs the steps as ONE sldg_step_n call (the x half-steps of consecutive steps in one pass).
--diagnostics adds sldg_diagnostics + sldg_moments after every step (the paper writes its invariants
every step), i.e. the "14 passes" accounting of its eq. (1).
Prints one JSON line.  Every step runs in the CUDA library; torch only builds the initial state.
"""
import argparse
import json

import numpy as np

from .. import workloads as W
from ..sldg import Sldg

NAMED = {"config1": W.CONFIG1, "config2": W.CONFIG2, "config3": W.CONFIG3, "config5": W.CONFIG5,
         "mixed13": W.MIXED13, "mixed23": W.MIXED23, "twostream": W.PAPER_TWOSTREAM}


def make_config(name, cells=None, order=None):
    cfg = NAMED[name]
    if cells is not None:
        cfg = cfg.scaled(cells, name=cfg.name + "-cells" + "x".join(str(c) for c in cells))
    if order is not None and order != cfg.order:
        cfg = W.Config(cfg.name + "-o%d" % order, cfg.dx, cfg.dv, cfg.cells, order, cfg.lo, cfg.hi, cfg.dt,
                       cfg.steps, cfg.kind, cfg.eps, cfg.k, dict(cfg.extra))
    return cfg


def device_initial_state(torch, s, cfg):
    """The separable analytic state f0 = outer(gv, gx) built on the device from the library's nodes."""
    coords = [s.node_coords(d) for d in range(cfg.dx + cfg.dv)]
    gx, gv = W.initial_factors(cfg, coords)
    f0 = torch.outer(torch.from_numpy(gv).cuda(), torch.from_numpy(gx).cuda()).reshape(-1).to(s.tdtype)
    s.set_initial(f0.contiguous())


def advect_group(s, base, cnt, tau):
    """The x- or v-group of one step through the public fused calls (what sldg_step issues)."""
    if cnt == 3:
        s.advect_triple(base, base + 1, base + 2, tau)
    elif cnt == 2:
        s.advect_pair(base, base + 1, tau)
    else:
        s.advect(base, tau)


def run(cfg, dtype="f64", steps=5, warmup=2, buckets=False, diagnostics=False, merged=False):
    import torch
    s = Sldg.from_config(cfg, dtype=dtype)
    device_initial_state(torch, s, cfg)
    names = ("advection_x", "compute_rho", "poisson", "advection_v")
    acc = {k: 0.0 for k in names}

    def one(ev):
        if not buckets:
            s.step(cfg.dt)
        else:
            marks = [torch.cuda.Event(enable_timing=True) for _ in range(6)]
            marks[0].record(); advect_group(s, 0, cfg.dx, 0.5 * cfg.dt)
            marks[1].record(); s.compute_rho(out=False)
            marks[2].record(); s.poisson_E(out=False)
            marks[3].record(); advect_group(s, cfg.dx, cfg.dx, cfg.dt)
            marks[4].record(); advect_group(s, 0, cfg.dx, 0.5 * cfg.dt)
            marks[5].record()
            if ev is not None:
                ev.append(marks)
        if diagnostics:
            return s.diagnostics() + s.moments()
        return None

    for _ in range(warmup):
        one(None)
    ev = []
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    l0 = s.launch_count()
    e0.record()
    last = None
    if merged and not buckets and not diagnostics:
        s.step_n(cfg.dt, steps)
    else:
        for _ in range(steps):
            last = one(ev)
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / steps
    for m in ev:
        acc["advection_x"] += m[0].elapsed_time(m[1]) + m[4].elapsed_time(m[5])
        acc["compute_rho"] += m[1].elapsed_time(m[2])
        acc["poisson"] += m[2].elapsed_time(m[3])
        acc["advection_v"] += m[3].elapsed_time(m[4])
    es = 8 if dtype == "f64" else 4
    passes = 2 * (2 * cfg.dx + cfg.dx) + 1 + (1 if diagnostics else 0)   # paper eq. (1) accounting
    mass, l2, ee = s.diagnostics()
    out = {"config": cfg.name, "cells": list(cfg.cells), "order": cfg.order, "dtype": dtype, "ndof": cfg.ndof,
           "steps": steps, "merged_half_steps": bool(merged), "ms_per_step": ms, "passes_paper_accounting": passes,
           "gbs_paper_eq1_style": passes * cfg.ndof * es / ms / 1e6,
           "launches_per_step": (s.launch_count() - l0) / steps,
           "mass": mass, "l2": l2, "electric_energy": ee}
    if buckets:
        out["buckets_ms_per_step"] = {k: v / steps for k, v in acc.items()}
    if last is not None:
        out["last_invariants"] = [float(x) if np.isscalar(x) else [float(y) for y in x] for x in last]
    s.close()
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--config", default="config3", choices=sorted(NAMED))
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=2)
    ap.add_argument("--dtype", default="f64", choices=["f64", "f32"])
    ap.add_argument("--order", type=int, default=None)
    ap.add_argument("--cells", default=None, help="comma-separated cell counts (default: the config's)")
    ap.add_argument("--buckets", action="store_true")
    ap.add_argument("--diagnostics", action="store_true")
    ap.add_argument("--merged", action="store_true")
    a = ap.parse_args()
    cells = tuple(int(c) for c in a.cells.split(",")) if a.cells else None
    cfg = make_config(a.config, cells, a.order)
    print(json.dumps(run(cfg, a.dtype, a.steps, a.warmup, a.buckets, a.diagnostics, a.merged)))


if __name__ == "__main__":
    main()
