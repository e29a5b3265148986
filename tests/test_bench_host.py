"""Host logic of bench.py's multi-GPU (replicas-only) path on CPU: world_size 2 over gloo.
Checks the max-over-ranks timing, the job-level aggregation and that only rank 0 runs the reference arm."""
import os
import socket
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    os.environ.update(RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1",
                      MASTER_PORT=str(port))
    sys.path.insert(0, ROOT)
    import torch
    import torch.distributed as dist

    import bench
    assert bench.dist_env() == (world, rank, rank)
    reduce_max, barrier = bench.dist_ops(world, "gloo", torch.device("cpu"))
    barrier()
    elapsed = 100.0 + 50.0 * rank                     # rank 1 is the slow replica
    agg = bench.aggregate_replicas(elapsed, k_steps=10, world=world, reduce_max=reduce_max)
    barrier()
    dist.destroy_process_group()
    q.put((rank, agg))


def test_replica_aggregation_world2_gloo():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    out = dict(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank in (0, 1):
        agg = out[rank]
        assert agg["ms_total"] == 150.0                         # max over ranks, on every rank
        assert agg["ms_per_step"] == 15.0
        assert agg["us_per_outer_job"] == pytest.approx(1e3 * 150.0 / (10 * 2))   # all ranks' iterations / max time


def test_single_rank_ops_are_identities():
    sys.path.insert(0, ROOT)
    import bench
    reduce_max, barrier = bench.dist_ops(1, "gloo", None)
    assert reduce_max(3.5) == 3.5 and barrier() is None
    agg = bench.aggregate_replicas(20.0, 4, 1, reduce_max)
    assert agg == dict(ms_total=20.0, ms_per_step=5.0, us_per_outer_job=5000.0)


def test_byte_model_matches_survey_table():
    """config 4, s = 4 -> MPK 14.388 GB, Gram 3.408 GB, update 7.602 GB, total 25.398 GB."""
    sys.path.insert(0, ROOT)
    import bench
    n, nnz = 320 ** 3, 7 * 320 ** 3 - 6 * 320 ** 2
    mb = bench.model_bytes(n, nnz, 4)
    assert round(mb["mpk"] / 1e9, 3) == 14.388 and round(mb["gram"] / 1e9, 3) == 3.408
    assert round(mb["update"] / 1e9, 3) == 7.602 and round(mb["total"] / 1e9, 3) == 25.398
    assert mb["spmv_per_launch"] * 4 == mb["mpk"]


def test_reference_arm_runs_on_rank0_only(monkeypatch):
    sys.path.insert(0, ROOT)
    import bench
    monkeypatch.setenv("RANK", "1")
    monkeypatch.setenv("WORLD_SIZE", "2")

    class A:
        grid, s, steps, warmup, gpus = 320, 4, 1, 1, 2
    assert bench.run_reference(A) is None


def test_ncu_traffic_table_is_read():
    """roofline.traffic comes from the committed ncu summary: SpMV rows of config 4, s = 4, launch-weighted."""
    sys.path.insert(0, ROOT)
    import bench
    t = bench.ncu_traffic(4, 4)
    n, nnz = 320 ** 3, 7 * 320 ** 3 - 6 * 320 ** 2
    alg = bench.model_bytes(n, nnz, 4)["spmv_per_launch"]
    assert t is not None and 0.95 * alg < t < 1.15 * alg          # measured DRAM traffic within 15 % of the algorithmic bytes
    assert bench.ncu_traffic(4, 3) is None and bench.ncu_traffic(9, 4) is None


def test_both_arms_print_the_same_workload_string():
    """`vs_reference.same_config` was false only because the two arms spelt config.workload differently."""
    import bench
    n, nnz = 320 ** 3, 7 * 320 ** 3 - 6 * 320 ** 2
    ours = bench.workload_string(4, 320, n, nnz, 4, "poisson7_320_sweep")
    ref = bench.workload_string(4, 320, n, nnz, 4)
    assert ours == ref and "320^3" in ours and f"nnz={nnz}" in ours and "s=4" in ours
    assert "config 2" in bench.workload_string(2, 128, 128 ** 3, 1, 4, "poisson7_128_s4")
