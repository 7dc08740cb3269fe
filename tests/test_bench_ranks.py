"""N > 1 plumbing of bench.py on CPU (gloo, world_size 2): the path has no data-path collective
(N ranks = N independent replicas), so what there is to check is the rank logic:
per-replica RHS, max-over-ranks timing, whole-job aggregation, and that the reference arm prints on
rank 0 only."""
import json
import os
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def _worker(rank, world, port, out):
    import torch.distributed as dist
    import bench
    from workloads import brick_mesh, rhs_unique
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    ms = bench.max_over_ranks(dist, [10.0 + 5.0 * rank, 3.0 - rank], "cpu")
    m = brick_mesh(2, 2, 2, 3, 0.05)
    f = rhs_unique(m, bench.replica_seed(1001, rank))
    dist.barrier()
    dist.destroy_process_group()
    out.put((rank, ms, float(f.sum())))


def test_gloo_two_ranks_max_and_replicas():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert res[0][1] == [15.0, 3.0] and res[1][1] == [15.0, 3.0]        # max over ranks, on every rank
    assert res[0][2] != res[1][2]                                       # each replica its own RHS


def test_whole_job_value_and_single_rank_identity():
    import bench
    assert bench.max_over_ranks(None, [1.5, 2.5], "cpu") == [1.5, 2.5]
    one = bench.whole_job_value(1e9, 4, 1, 100.0)
    assert one == pytest.approx(40.0)
    assert bench.whole_job_value(1e9, 4, 8, 100.0) == pytest.approx(8 * one)
    assert bench.replica_seed(1005, 0) == 1005 and bench.replica_seed(1005, 3) != bench.replica_seed(1005, 2)


def test_reference_arm_prints_on_rank0_only():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--steps", "1", "--warmup", "0", "--workload", "config1"],
                       capture_output=True, text=True, env=env, timeout=300)
    assert r.returncode == 0 and r.stdout.strip() == ""
    env["RANK"] = "0"
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--steps", "1", "--warmup", "0", "--workload", "config1"],
                       capture_output=True, text=True, env=env, timeout=300)
    line = json.loads(r.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["n_gpus"] == 2 and line["gpu_launches"] == 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["e2e"]["h2d_bytes_per_step"] == 0
    assert np.isfinite(line["value"]) and line["value"] > 0
