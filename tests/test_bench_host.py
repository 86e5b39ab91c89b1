"""Host-side logic of bench.py that needs no GPU: the replicas-only aggregation over ranks
(world_size 2, gloo, 127.0.0.1), the traffic table, and the reference arm's JSON line."""
import csv
import json
import os
import socket
import subprocess
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
import bench  # noqa: E402


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    # rank r measured (total, apply, e2e, solve) = base * (1 + r): the job's time is the slowest rank's
    got = bench.max_over_ranks([10.0 * (1 + rank), 2.0 * (1 + rank), 4.0 * (1 + rank), 0.1 * (1 + rank)], dist, "cpu")
    dist.barrier()
    dist.destroy_process_group()
    q.put((rank, got))


def test_max_over_ranks_gloo_world2():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    ps = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in ps:
        p.start()
    res = dict(q.get(timeout=120) for _ in ps)
    for p in ps:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert res[0] == res[1] == [20.0, 4.0, 8.0, 0.2]
    # two replicas, each 16 GB in 4 ms -> 8 TB/s whole-job
    assert abs(bench.aggregate_value(2, 16e9, 4.0) - 8000.0) < 1e-9


def test_single_rank_passthrough():
    assert bench.max_over_ranks([1.5, 2.5], None, "cpu") == [1.5, 2.5]


def test_traffic_table_parses():
    rows = list(csv.DictReader(open(os.path.join(ROOT, "profiles", "apply_ncu_traffic.csv"))))
    assert rows and all(set(r) >= {"workload", "kernel", "dram_bytes_per_launch"} for r in rows)
    for r in rows:
        alg = 512000 * bench.alg_bytes_per_site(4, 1)
        if r["workload"] == "20x20x20x64-fp32":
            assert 0.95 * alg < int(r["dram_bytes_per_launch"]) < 1.2 * alg


def test_reference_arm_prints_contract_line():
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "1", "--warmup", "0",
                          "--workload", "4x4x4x8-fp64"], capture_output=True, text=True, timeout=300)
    assert out.returncode == 0, out.stderr
    line = json.loads(out.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["cpu_baseline"]["kind"] == "oracle"
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["value"] > 0
