"""The N>1 path of bench.py is "replicas only": no data-path collective, only
a MAX over ranks of the timings and distinct seeds per rank.  Covered here with world_size 2 on gloo."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    import bench
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    mine = [10.0 + rank, 5.0 - rank, 7.0]
    red = bench.reduce_max_over_ranks(mine)
    dist.barrier()
    dist.destroy_process_group()
    with open(f"{out}.{rank}", "w") as f:
        json.dump({"red": red, "seeds": bench.replica_seeds(3, rank)}, f)


def test_max_over_ranks_and_replica_seeds(tmp_path):
    import torch.multiprocessing as mp
    out = str(tmp_path / "r")
    mp.spawn(_worker, args=(2, 29611, out), nprocs=2, join=True)
    r = [json.load(open(f"{out}.{k}")) for k in range(2)]
    assert r[0]["red"] == r[1]["red"] == [11.0, 5.0, 7.0]
    assert r[0]["seeds"] != r[1]["seeds"] and r[0]["seeds"] == [1003, 2003]


def test_aggregate_rate_counts_every_replica():
    sys.path.insert(0, ROOT)
    import bench
    one = bench.aggregate_cholesky_gflops(32768, 1, 400.0)
    assert abs(one - 32768 ** 3 / 3 / 0.4 / 1e9) < 1e-6
    assert abs(bench.aggregate_cholesky_gflops(32768, 8, 400.0) - 8 * one) < 1e-6
    assert bench.reduce_max_over_ranks([1.0, 2.0]) == [1.0, 2.0]      # no process group: identity


def test_reference_arm_under_torchrun_prints_one_line():
    """--impl reference with 2 ranks: rank 0 alone runs the oracle and prints; rank 1 exits 0."""
    env = dict(os.environ, OMP_NUM_THREADS="4")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr", "127.0.0.1",
           "--master-port", "29612", os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1",
           "--warmup", "0", "--config", "1"]
    r = subprocess.run(cmd, capture_output=True, text=True, timeout=600, env=env, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [json.loads(l) for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = lines[0]
    assert d["impl"] == "reference" and d["value"] > 0 and d["unit"] == "GFLOP/s"
    assert d["cpu_baseline"]["kind"] == "oracle" and d["e2e"]["h2d_bytes_per_step"] == 0
    assert d["e2e"]["unit"] == "GFLOP/s" == sys.modules.get("bench", __import__("bench")).E2E_UNIT
    # config 1 is small enough for the oracle to run the config itself: the workload string is not a sample
    assert d["config"]["workload"].startswith("c1:") and "sample_n" not in d["config"]


def test_reference_arm_names_the_sample_it_runs():
    sys.path.insert(0, ROOT)
    import bench
    from paper_2602_19683_b200 import nfir
    n, m, sampled = bench.reference_sample(nfir.CONFIGS[3])
    assert sampled and (n, m) == bench.ORACLE_SAMPLE
    assert bench.reference_sample(nfir.CONFIGS[0]) == (128, 128, False)
