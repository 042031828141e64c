#!/usr/bin/env python
"""bench.py -- SLDG hot path on B200: one JSON line.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload NAME]

A "step" is one pass of the whole hot path over the config-4
workload (BASELINE.json configs[3]: 2+2 D, 128^2 x 64^2 cells, o = 3, seeded uniform f, per-cell
seeded shifts), fp64:
    translate x_1, translate x_2 (a-1 + a-2) -> rho (a-3) -> Poisson/E (a-4)
    -> translate v_1, translate v_2 (a-1 + a-2) -> diagnostics (a-6: rho + s2 + Poisson + scalars)
`value` = achieved HBM GB/s per translation sweep = 2*N*sizeof(T) * (#sweeps) / (time spent in the
sweeps), timed with CUDA events on the launching stream inside the timed steps; `ms_per_step` is the
whole step.  N > 1: independent replicas, one per GPU ("replicas only"), value = sum.
"""
import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_1907_08316_b200 import workloads as W  # noqa: E402

TRAFFIC_TABLE = os.path.join(ROOT, "profiles", "traffic_launches_r3.md")


def traffic_bytes(workload, dtype):
    """{dim: dram__bytes_read.sum + dram__bytes_write.sum per launch} of the sweep kernel of each direction, parsed
    from the table of the ncu capture of this very command at full size (profiles/traffic_launches_r3.md: rows
    `| <workload> | <dtype> | dim<k> | kernel | read GB | write GB | ...`); {} where nothing was captured."""
    out = {}
    try:
        with open(TRAFFIC_TABLE) as fh:
            for row in fh:
                cells = [c.strip() for c in row.strip().strip("|").split("|")]
                if len(cells) >= 6 and cells[0] == workload and cells[1] == dtype and cells[2].startswith("dim"):
                    out[int(cells[2][3:])] = (float(cells[4]) + float(cells[5])) * 1e9
    except (OSError, ValueError):
        return {}
    return out


METRIC = "achieved_hbm_gbs_per_translation_sweep"
UNIT = "GB/s"


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as fh:
            return float(json.load(fh)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """nvidia-smi clocks/throttle reasons sampled DURING the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.proc, self.path = index, None, None

    def start(self):
        try:
            fd, self.path = tempfile.mkstemp(suffix=".csv")
            os.close(fd)
            self.fh = open(self.path, "w")
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                 "--format=csv,noheader,nounits", "-lms", "100"], stdout=self.fh, stderr=subprocess.DEVNULL)
        except Exception:
            self.proc = None

    def stop(self, full=False):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": []}
        if self.proc is None:
            return out
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        self.fh.close()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in open(self.path):
            p = [x.strip() for x in line.split(",")]
            if len(p) < 7:
                continue
            try:
                sm.append(float(p[0])); mx.append(float(p[1]))
            except ValueError:
                continue
            for n, v in zip(names, p[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        os.unlink(self.path)
        if sm:
            out = {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(mx)), "reasons": sorted(reasons),
                   "samples": len(sm)}
            if full:
                out["sm_mhz_min"] = float(min(sm)); out["sm_mhz_peak"] = float(max(sm))
        return out


# ---------------------------------------------------------------------------------------------
# workloads
# ---------------------------------------------------------------------------------------------
def pick_workload(name):
    """config4 (default, the configuration the metric is quoted on) or a reduced twin 'config4/2',
    'config4/4' (every n_d divided) for boxes where the full size does not fit."""
    if "/" in name:
        base, div = name.split("/")
        cfg = W.CONFIGS[base]
        cells = tuple(max(1, c // int(div)) for c in cfg.cells)
        return cfg.scaled(cells, name=cfg.name + "/" + div)
    return W.CONFIGS[name]


def step_bytes(cfg, esize):
    """Algorithmic HBM bytes of one bench step: 2(dx+dv)... here 4 sweeps (1R+1W) + 2 reads of f."""
    D = cfg.dx + cfg.dv
    return (2 * D + 2) * cfg.ndof * esize


# ---------------------------------------------------------------------------------------------
# the CPU oracle timed on the host cores (cpu_baseline leg and --impl reference)
# ---------------------------------------------------------------------------------------------
def oracle_step_factory(cfg, dtype):
    from oracle import sldg_oracle as O
    npdt = np.float64 if dtype == "f64" else np.float32
    g = O.Grid(cfg.dx, cfg.dv, cfg.cells, cfg.order, cfg.lo, cfg.hi)
    D = cfg.dx + cfg.dv
    f = np.empty(cfg.ndof, dtype=npdt)
    chunk = 1 << 24
    for a in range(0, cfg.ndof, chunk):          # chunked: bounded temporaries
        b = min(cfg.ndof, a + chunk)
        f[a:b] = W.uniform(W.SEED, W.TAG_F, np.arange(a, b, dtype=np.uint64)).astype(npdt)
    shifts = [W.config4_shifts(cfg, d) for d in range(D)]
    deps = [[cfg.dx + d] if d < cfg.dx else list(range(cfg.dx)) for d in range(D)]

    per_dim = {d: 0.0 for d in range(D)}      # seconds spent in the sweeps of each direction (all steps)

    def step():
        t_sweeps = 0.0
        for d in range(cfg.dx):
            t0 = time.perf_counter()
            O.translate(f, cfg.N, cfg.order, d, shifts[d], deps[d])
            dt_ = time.perf_counter() - t0
            t_sweeps += dt_; per_dim[d] += dt_
        rho = g.rho(f)
        g.poisson_E(rho)
        for d in range(cfg.dx, D):
            t0 = time.perf_counter()
            O.translate(f, cfg.N, cfg.order, d, shifts[d], deps[d])
            dt_ = time.perf_counter() - t0
            t_sweeps += dt_; per_dim[d] += dt_
        g.diagnostics(f)
        return t_sweeps

    step.per_dim = per_dim
    return step, O.num_threads()


def choose_oracle_sample(total_steps, budget_s=120.0):
    """Largest reduced twin of config 4 whose `total_steps` oracle steps fit the time budget."""
    from oracle import sldg_oracle as O
    probe = W.CONFIG4.scaled((32, 32, 16, 16))
    f = np.random.default_rng(0).random(probe.ndof)
    sig = W.config4_shifts(probe, 2)
    O.translate(f, probe.N, probe.order, 2, sig, [0, 1])
    t0 = time.perf_counter()
    O.translate(f, probe.N, probe.order, 2, sig, [0, 1])
    rate = probe.ndof / (time.perf_counter() - t0)          # DOF updates / s, whole machine
    for cells in ((64, 64, 32, 32), (32, 32, 32, 32), (32, 32, 16, 16), (16, 16, 16, 16)):
        cfg = W.CONFIG4.scaled(cells)
        est = total_steps * 6.0 * cfg.ndof / rate + 25.0 * cfg.ndof / 3.4e8
        if est <= budget_s:
            return cfg
    return W.CONFIG4.scaled((16, 16, 8, 8))


def cpu_model():
    try:
        for line in open("/proc/cpuinfo"):
            if line.startswith("model name"):
                return line.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


_ONE_THREAD_SNIPPET = r"""
import sys, time, numpy as np
sys.path.insert(0, %r)
from oracle import sldg_oracle as O
from paper_1907_08316_b200 import workloads as W
cfg = W.CONFIG4.scaled((32, 32, 16, 16))
f = np.random.default_rng(0).random(cfg.ndof)
D = cfg.dx + cfg.dv
t = 0.0
for d in range(D):
    sig = W.config4_shifts(cfg, d)
    dep = [cfg.dx + d] if d < cfg.dx else list(range(cfg.dx))
    t0 = time.perf_counter(); O.translate(f, cfg.N, cfg.order, d, sig, dep); t += time.perf_counter() - t0
print(O.num_threads(), cfg.ndof * D / t)
"""


def oracle_one_thread():
    """The same oracle with OMP_NUM_THREADS=1 on a small twin (one sweep per direction): DOF updates/s."""
    env = dict(os.environ, OMP_NUM_THREADS="1")
    try:
        out = subprocess.run([sys.executable, "-c", _ONE_THREAD_SNIPPET % ROOT], env=env, capture_output=True,
                             text=True, timeout=120).stdout.split()
        return {"threads": int(out[0]), "dof_updates_per_s": float(out[1]),
                "value": 2.0 * 8 * float(out[1]) / 1e9, "unit": UNIT,
                "sample": "one sweep per direction, config-4 recipe, cells=(32, 32, 16, 16)"}
    except Exception as exc:
        return {"error": str(exc)}


def oracle_config3_step():
    """One full-size Strang step of config 3 by the oracle (seconds), S:8(d)."""
    from oracle import sldg_oracle as O
    cfg = W.CONFIG3
    g = O.Grid(cfg.dx, cfg.dv, cfg.cells, cfg.order, cfg.lo, cfg.hi)
    f = W.initial_state(cfg, [g.coords(d) for d in range(cfg.dx + cfg.dv)])
    t0 = time.perf_counter()
    g.step(f, cfg.dt)
    return time.perf_counter() - t0


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    total = args.steps + args.warmup
    cfg = choose_oracle_sample(total, budget_s=150.0)
    step, cores = oracle_step_factory(cfg, "f64")
    for _ in range(args.warmup):
        step()
    t0 = time.perf_counter()
    t_sw = 0.0
    for _ in range(args.steps):
        t_sw += step()
    wall = time.perf_counter() - t0
    D = cfg.dx + cfg.dv
    value = 2.0 * cfg.ndof * 8 * D * args.steps / t_sw / 1e9
    sample = "config-4 recipe on reduced twin cells=%s (%.2e DOF), full bench step per step" % (cfg.cells, cfg.ndof)
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * wall / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic", "config": {"workload": W.CONFIG4.name, "sample": sample},
        "dof_updates_per_s": cfg.ndof * D * args.steps / t_sw,
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


# ---------------------------------------------------------------------------------------------
# our arm: the CUDA library through its Python binding (C-ABI calls only)
# ---------------------------------------------------------------------------------------------
def host_mem_available_bytes():
    try:
        for line in open("/proc/meminfo"):
            if line.startswith("MemAvailable:"):
                return int(line.split()[1]) * 1024
    except OSError:
        pass
    return 0


def sweep_table(torch, s, cfg, dtype, reps, warm):
    """Per-direction sweep timings (ms, median) of one solver with the config's own shift recipe."""
    D = cfg.dx + cfg.dv
    es = 8 if dtype == "f64" else 4
    out = {}
    for dim in range(D):
        if cfg.kind == "uniform":
            sig = W.config4_shifts(cfg, dim)
        else:   # physics-like: x-shifts from v dt/2/h, v-shifts |sigma| << 1 (seeded)
            cnt = cfg.N[cfg.dx + dim] if dim < cfg.dx else cfg.X
            if dim < cfg.dx:
                va = cfg.dx + dim
                h = (cfg.hi[dim] - cfg.lo[dim]) / cfg.cells[dim]
                sig = np.linspace(cfg.lo[va], cfg.hi[va], cnt) * 0.5 * cfg.dt / h
            else:
                sig = 0.02 * (W.uniform(W.SEED, W.TAG_SHIFT + dim, np.arange(cnt, dtype=np.uint64)) - 0.5)
        sd = torch.from_numpy(np.ascontiguousarray(sig)).cuda()
        for _ in range(warm):
            s.translate(dim, sd)
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(reps + 1)]
        ev[0].record()
        for r in range(reps):
            s.translate(dim, sd)
            ev[r + 1].record()
        torch.cuda.synchronize()
        ts = [ev[i].elapsed_time(ev[i + 1]) for i in range(reps)]
        t = float(np.median(ts))
        out["dim%d" % dim] = {"ms": t, "gbs": 2 * cfg.ndof * es / t / 1e6, "dof_per_s": cfg.ndof / t * 1e3,
                              "best_ms": float(min(ts))}
    return out


def strang_step_table(torch, Sldg, cfg, dtype, steps):
    """Full Strang steps (sldg_step, fused sweep pairs) of a Landau config: ms per step and the
    paper's eq. (1) style bandwidth (2(2dx+dx)+1 passes of N*sizeof(T) per step)."""
    s = Sldg.from_config(cfg, dtype=dtype)
    coords = [s.node_coords(d) for d in range(cfg.dx + cfg.dv)]
    gx, gv = W.initial_factors(cfg, coords)
    f0 = torch.outer(torch.from_numpy(gv).cuda(), torch.from_numpy(gx).cuda()).reshape(-1).to(s.tdtype)
    s.set_initial(f0.contiguous())
    del f0
    for _ in range(3):
        s.step(cfg.dt)
    e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
    l0 = s.launch_count()
    e0.record()
    for _ in range(steps):
        s.step(cfg.dt)
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / steps
    launches_per_step = (s.launch_count() - l0) / steps
    # the same steps with the x half-steps of consecutive steps merged into one pass (sldg_step_n; same f)
    e2 = torch.cuda.Event(enable_timing=True); e3 = torch.cuda.Event(enable_timing=True)
    s.step_n(cfg.dt, 2)
    e2.record()
    s.step_n(cfg.dt, steps)
    e3.record()
    torch.cuda.synchronize()
    ms_merged = e2.elapsed_time(e3) / steps
    # the paper's own loop writes the invariants once per step: one more read of f (sldg_invariants)
    # (CUDA events on the launching stream, as everywhere else; sldg_invariants synchronises once per call to hand
    # its scalars to the host, which is part of what the loop costs)
    s.step(cfg.dt); s.invariants()
    e4 = torch.cuda.Event(enable_timing=True); e5 = torch.cuda.Event(enable_timing=True)
    e4.record()
    for _ in range(steps):
        s.step(cfg.dt)
        s.invariants()
    e5.record()
    torch.cuda.synchronize()
    ms_inv = e4.elapsed_time(e5) / steps
    es = 8 if dtype == "f64" else 4
    passes = 2 * (3 * cfg.dx) + 1
    mass, l2, ee = s.diagnostics()
    out = {"ms_per_step": ms, "ms_per_step_merged_half_steps": ms_merged,
           "gbs_paper_eq1_style_merged": passes * cfg.ndof * es / ms_merged / 1e6,
           "ms_per_step_with_invariants_every_step": ms_inv, "passes_paper_accounting": passes,
           "gbs_paper_eq1_style_with_invariants": (passes + 1) * cfg.ndof * es / ms_inv / 1e6,
           "gbs_paper_eq1_style": passes * cfg.ndof * es / ms / 1e6,
           "dof_updates_per_s": 3 * cfg.dx * cfg.ndof / ms * 1e3,
           "launches_per_step": launches_per_step, "mass": mass, "electric_energy": ee}
    s.close()
    del s
    torch.cuda.empty_cache()
    return out


def max_over_ranks(values, world, device):
    """Element-wise MAX of a list of floats over all ranks (timings are max-over-ranks)."""
    if world <= 1:
        return [float(v) for v in values]
    import torch
    import torch.distributed as dist
    t = torch.tensor(list(values), dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(x) for x in t]


def replica_throughput(world, bytes_per_replica, ms_max):
    """Whole-job GB/s of `world` independent replicas that each moved bytes_per_replica in ms_max."""
    return world * bytes_per_replica / ms_max / 1e6


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_1907_08316_b200.sldg import Sldg

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the SLDG library has no CPU path "
                         "(use --impl reference for the oracle timing)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    cfg = pick_workload(args.workload)
    dtype = args.dtype
    es = 8 if dtype == "f64" else 4
    D = cfg.dx + cfg.dv
    peak, peak_src = measured_peaks()

    s = Sldg.from_config(cfg, dtype=dtype, device="cuda:%d" % local)
    s.fill_uniform(W.SEED + rank, W.TAG_F)
    shifts = [torch.from_numpy(W.config4_shifts(cfg, d)).cuda() for d in range(D)]

    def step(events=None):
        for d in range(cfg.dx):
            if events is not None:
                e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
                e0.record(); s.translate(d, shifts[d]); e1.record(); events.append((d, e0, e1))
            else:
                s.translate(d, shifts[d])
        s.compute_rho(out=False)
        s.poisson_E(out=False)
        for d in range(cfg.dx, D):
            if events is not None:
                e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
                e0.record(); s.translate(d, shifts[d]); e1.record(); events.append((d, e0, e1))
            else:
                s.translate(d, shifts[d])
        return s.diagnostics()

    for _ in range(args.warmup):
        step()
    sampler = ClockSampler(local)
    barrier()
    sampler.start()
    events = []
    l0 = s.launch_count()
    t_start = torch.cuda.Event(enable_timing=True); t_end = torch.cuda.Event(enable_timing=True)
    barrier()
    t_start.record()
    for _ in range(args.steps):
        step(events)
    t_end.record()
    barrier()
    clocks = sampler.stop()
    launches = s.launch_count() - l0
    total_ms = t_start.elapsed_time(t_end)
    per_dim = {d: [] for d in range(D)}
    for d, e0, e1 in events:
        per_dim[d].append(e0.elapsed_time(e1))
    sweep_ms = sum(sum(v) for v in per_dim.values())
    nsweeps = sum(len(v) for v in per_dim.values())
    total_ms, sweep_ms = max_over_ranks([total_ms, sweep_ms], world, "cuda")
    sweep_bytes = 2.0 * cfg.ndof * es
    value = replica_throughput(world, sweep_bytes * nsweeps, sweep_ms)   # GB/s per sweep, all replicas
    # dominant kernel = slowest direction's sweep kernel
    dim_avg = {d: float(np.mean(v)) for d, v in per_dim.items()}
    dom = max(dim_avg, key=dim_avg.get)
    roofline = {"bound": "hbm", "achieved": sweep_bytes / dim_avg[dom] / 1e6, "peak": peak, "unit": "GB/s",
                "frac": sweep_bytes / dim_avg[dom] / 1e6 / peak,
                "traffic": traffic_bytes(cfg.name, dtype).get(dom),
                "traffic_source": "ncu dram__bytes_read.sum + dram__bytes_write.sum per launch, parsed from profiles/traffic_launches_r3.md",
                "kernel": "translation sweep along dim %d (slowest direction)" % dom,
                "algorithmic_bytes_per_launch": sweep_bytes, "peak_source": peak_src,
                "per_direction_gbs": {"dim%d" % d: sweep_bytes / t / 1e6 for d, t in dim_avg.items()},
                "frac_of_8000_nominal": sweep_bytes / dim_avg[dom] / 1e6 / 8000.0}

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": total_ms / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": dtype, "data": "synthetic",
        "config": {"workload": cfg.name, "cells": list(cfg.cells), "order": cfg.order, "ndof": cfg.ndof,
                   "bytes_per_copy_of_f": cfg.ndof * es, "parallelism": "replicas x%d" % world,
                   "l2_policy": "inputs larger than L2 (%.1f GB per copy of f vs 126 MB)" % (cfg.ndof * es / 1e9),
                   "step": "translate x1,x2 -> rho -> poisson -> translate v1,v2 -> diagnostics"},
        "dof_updates_per_s": world * cfg.ndof * nsweeps / sweep_ms * 1e3,
        "step_gbs_paper_eq1_style": world * step_bytes(cfg, es) / (total_ms / args.steps) / 1e6,
        "roofline": roofline, "clocks": clocks, "gpu_launches": int(launches),
    }

    # ---- per-direction SM clock (min / median / max) while that direction's sweep runs alone, S:8(d)
    if world == 1:
        pdc = {}
        for d in range(D):
            smp = ClockSampler(local)
            torch.cuda.synchronize()
            smp.start()
            e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
            nrep = 40
            e0.record()
            for _ in range(nrep):
                s.translate(d, shifts[d])
            e1.record()
            torch.cuda.synchronize()
            ck = smp.stop(full=True)
            pdc["dim%d" % d] = {"sm_mhz_min": ck.get("sm_mhz_min"), "sm_mhz": ck.get("sm_mhz"),
                                "sm_mhz_max": ck.get("sm_mhz_peak"), "reasons": ck.get("reasons"),
                                "gbs_alone": sweep_bytes * nrep / e0.elapsed_time(e1) / 1e6}
        roofline["per_direction_clocks"] = pdc

    # ---- e2e: the same step through the C-ABI with HOST buffers (pinned), copies inside the timing
    if rank == 0 or world > 1:
        nbytes = cfg.ndof * es
        e2e_cfg, e2e_note = cfg, "full workload"
        if host_mem_available_bytes() < 2.5 * nbytes:
            e2e_note = "host RAM too small for a pinned copy of f; e2e not measured"
            line["e2e"] = {"value": None, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0,
                           "note": e2e_note}
        else:
            hbuf = torch.empty(cfg.ndof, dtype=s.tdtype, pin_memory=True)
            s.get_f(hbuf)
            k = max(1, min(args.steps, 2))
            s.set_initial(hbuf); step(); s.get_f(hbuf)          # warm
            barrier()
            t0 = time.perf_counter()
            for _ in range(k):
                s.set_initial(hbuf)
                step()
                s.get_f(hbuf)
            torch.cuda.synchronize()
            dt = time.perf_counter() - t0
            dt = max_over_ranks([dt], world, "cuda")[0]
            line["e2e"] = {"value": world * sweep_bytes * D * k / dt / 1e9, "unit": UNIT,
                           "h2d_bytes_per_step": nbytes, "d2h_bytes_per_step": nbytes + 24,
                           "ms_per_step": 1e3 * dt / k, "steps": k, "note": e2e_note +
                           "; per step: sldg_set_initial(host) + bench step + sldg_get_f(host)"}
            del hbuf

    # ---- fp32 and the other roofline configs, per direction (rank 0 of a 1-GPU run only)
    if world == 1 and not args.no_extras:
        extras = {}
        s.close(); del s; torch.cuda.empty_cache()
        for name, dt_ in (("config4", "f32"), ("config3", "f64"), ("config5", "f64")):
            c2 = W.CONFIGS[name] if args.workload == "config4" else pick_workload(name + "/2")
            try:
                s2 = Sldg.from_config(c2, dtype=dt_)
                s2.fill_uniform(W.SEED, W.TAG_F)
                extras["%s-%s" % (c2.name, dt_)] = sweep_table(torch, s2, c2, dt_, reps=10, warm=3)
                s2.close(); del s2; torch.cuda.empty_cache()
            except Exception as exc:        # report, never hide
                extras["%s-%s" % (c2.name, dt_)] = {"error": str(exc)}
        if args.workload == "config4":
            # the paper's order axis (Fig. 2: bandwidth at o = 2, 4, 6): single sweeps of the 2+2 D two-stream
            # set-up at o = 4, 5, 6 on 3.3e9 DOF each (60^4, 48^4, 40^4 cells), physics-like shifts
            for o_, n_ in ((4, 60), (5, 48), (6, 40)):
                base = W.PAPER_TWOSTREAM
                c2 = W.Config("order-axis-2+2-o%d" % o_, 2, 2, (n_,) * 4, o_, base.lo, base.hi, dt=base.dt,
                              kind=base.kind, eps=base.eps, k=base.k, extra=dict(base.extra))
                try:
                    s2 = Sldg.from_config(c2, dtype="f64")
                    s2.fill_uniform(W.SEED, W.TAG_F)
                    extras["%s-f64" % c2.name] = sweep_table(torch, s2, c2, "f64", reps=10, warm=3)
                    s2.close(); del s2; torch.cuda.empty_cache()
                except Exception as exc:
                    extras["%s-f64" % c2.name] = {"error": str(exc)}
        line["sweeps_other_configs"] = extras
        steps_tab = {}
        for name, nst in (("config3", 20), ("config5", 5)):
            c2 = W.CONFIGS[name] if args.workload == "config4" else pick_workload(name + "/2")
            try:
                steps_tab[c2.name] = strang_step_table(torch, Sldg, c2, "f64", nst)
            except Exception as exc:
                steps_tab[c2.name] = {"error": str(exc)}
        if args.workload == "config4":          # the paper's own set-ups, context only: its section-7 mixed dimensions
            # (1+3 D, 2+3 D at o = 4) and its headline 2+2 D run at o = 4 (60^4 cells, eq. (2); 470 GB/s on a V100)
            for c2 in (W.MIXED13, W.MIXED23, W.PAPER_TWOSTREAM):
                try:
                    steps_tab[c2.name] = strang_step_table(torch, Sldg, c2, "f64", min(c2.steps, 5) if c2.steps else 5)
                except Exception as exc:
                    steps_tab[c2.name] = {"error": str(exc)}
        line["strang_steps_fused"] = steps_tab

    # ---- the oracle on the host cores, bounded sample (rank 0, N = 1 only)
    if world == 1 and rank == 0 and not args.no_cpu_baseline:
        ocfg = choose_oracle_sample(2, budget_s=30.0)
        ostep, cores = oracle_step_factory(ocfg, dtype)
        nrep, t_sw, t0 = 0, 0.0, time.perf_counter()
        while nrep < 4 and (nrep == 0 or time.perf_counter() - t0 < 12.0):     # ~10-20 s of CPU work
            t_sw += ostep()
            nrep += 1
        line["cpu_baseline"] = {
            "value": 2.0 * ocfg.ndof * es * D * nrep / t_sw / 1e9, "unit": UNIT, "cores": cores, "kind": "oracle",
            "dof_updates_per_s": ocfg.ndof * D * nrep / t_sw,
            "per_direction_gbs": {"dim%d" % d: 2.0 * ocfg.ndof * es * nrep / t / 1e9 for d, t in ostep.per_dim.items()},
            "sample": "%d bench step(s) of the config-4 recipe on reduced twin cells=%s (%.2e DOF)" % (nrep, ocfg.cells, ocfg.ndof),
            "cpu_model": cpu_model(), "one_thread": oracle_one_thread()}
        try:        # S:8(d): the oracle's full-size config-3 Strang step beside the library's
            t_or = oracle_config3_step()
            gpu_ms = line.get("strang_steps_fused", {}).get(W.CONFIG3.name, {}).get("ms_per_step")
            line["cpu_baseline"]["config3_step"] = {"oracle_ms": 1e3 * t_or, "gpu_ms": gpu_ms, "cores": cores}
        except Exception as exc:
            line["cpu_baseline"]["config3_step"] = {"error": str(exc)}

    if rank == 0:
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="config4")
    ap.add_argument("--dtype", default="f64", choices=["f64", "f32"])
    ap.add_argument("--no-extras", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
