"""CPU, world_size 2, gloo: the N > 1 host logic of bench.py ("replicas only"):
timings are reduced with MAX over ranks, the whole-job value is the sum over replicas, and only
rank 0 of the reference arm does work."""
import json
import os
import socket
import subprocess
import sys

import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, out):
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    import bench
    dist.init_process_group("gloo", init_method="tcp://127.0.0.1:%d" % port, rank=rank, world_size=world)
    # rank r pretends its timed region took (10 + 5 r) ms in total and (8 + r) ms in the sweeps
    total, sweeps = bench.max_over_ranks([10.0 + 5.0 * rank, 8.0 + rank], world, "cpu")
    val = bench.replica_throughput(world, 1e9, sweeps)
    dist.barrier()
    if rank == 0:
        out.put((total, sweeps, val))
    dist.destroy_process_group()


def test_max_over_ranks_and_replica_sum_world2():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    total, sweeps, val = q.get(timeout=120)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert total == 15.0 and sweeps == 9.0            # MAX over ranks, not rank 0's own 10 / 8
    assert abs(val - 2 * 1e9 / 9.0 / 1e6) < 1e-9       # two replicas' bytes over the slowest rank's time


def test_single_rank_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks([3.0, 4.0], 1, "cpu") == [3.0, 4.0]
    assert bench.replica_throughput(1, 2e9, 1.0) == 2000.0


def test_reference_arm_only_rank0_prints():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--steps", "1", "--warmup", "0"], env=env, capture_output=True, text=True, timeout=120)
    assert r.returncode == 0 and r.stdout.strip() == ""


def test_reference_arm_json_contract():
    """bench.py --impl reference (the oracle on the host cores) prints ONE JSON line with the contract keys."""
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "1",
                        "--warmup", "0"], capture_output=True, text=True, timeout=600)
    assert r.returncode == 0, r.stderr[-500:]
    lines = [ln for ln in r.stdout.splitlines() if ln.strip()]
    assert len(lines) == 1
    d = json.loads(lines[0])
    for key in ("impl", "metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better",
                "scaling", "vs_baseline", "dtype", "data", "config", "cpu_baseline", "e2e", "gpu_launches"):
        assert key in d, key
    assert d["impl"] == "reference" and d["unit"] == "GB/s" and d["value"] > 0 and d["vs_baseline"] is None
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] >= 1
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and "workload" in d["config"]


def test_roofline_traffic_is_parsed_from_the_profile_table():
    """bench.py carries no typed-in DRAM byte counts: roofline.traffic comes from the ncu table under profiles/."""
    import bench
    t = bench.traffic_bytes("config4-sweep-2+2", "f64")
    assert sorted(t) == [0, 1, 2, 3]
    algorithmic = 2 * 5435817984 * 8
    for d, b in t.items():
        assert 0.99 * algorithmic <= b <= 1.02 * algorithmic, (d, b)     # no kernel re-reads f
    assert bench.traffic_bytes("no-such-workload", "f64") == {}
