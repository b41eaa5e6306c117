"""The N > 1 path of bench.py on CPU: two gloo ranks (world_size 2, 127.0.0.1).  The SP2 path does not shard
(replicas only), so the only cross-rank step is the MAX over ranks of the per-rank timings; rank 0 alone
prints the JSON line."""
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
    sys.path.insert(0, ROOT)
    import torch.distributed as dist

    import bench

    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    # every rank reports a different time: the job time is the slowest replica's
    mine = [10.0 + rank, 20.0 - rank]
    out = bench.aggregate_over_ranks(mine, dist, None)
    dist.barrier()
    dist.destroy_process_group()
    q.put((rank, out))


def test_max_over_ranks_world_size_2():
    import torch.multiprocessing as mp

    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    got = dict(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert got[0] == got[1] == [11.0, 20.0]


def test_single_process_aggregation_and_replica_throughput():
    sys.path.insert(0, ROOT)
    import bench

    assert bench.aggregate_over_ranks([1.5, 2.5]) == [1.5, 2.5]
    assert bench.replicas_per_second(8, 5.0) == pytest.approx(1600.0)


def test_reference_arm_runs_on_rank0_only(monkeypatch, capsys):
    """--impl reference under torchrun: ranks other than 0 exit 0 without work."""
    sys.path.insert(0, ROOT)
    import bench

    monkeypatch.setenv("RANK", "1")

    class A:
        workload, steps, warmup, gpus = "dense_n256", 1, 0, 2

    assert bench.run_reference(A) == 0
    assert capsys.readouterr().out == ""


@pytest.mark.parametrize("workload,metric", [("dense_n256", "sp2_time_to_D_ms"), ("cheby_n500", "chebyshev_time_to_D_ms")])
def test_reference_arm_prints_the_contract_line(monkeypatch, capsys, workload, metric):
    """--impl reference on rank 0 (no GPU needed: it times the oracle): one JSON line with the reference-arm keys."""
    import json

    sys.path.insert(0, ROOT)
    import bench

    monkeypatch.setenv("RANK", "0")

    class A:
        steps, warmup, gpus = 1, 0, 1

    A.workload = workload
    assert bench.run_reference(A) == 0
    lines = [l for l in capsys.readouterr().out.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["metric"] == metric and d["unit"] == "ms" and d["value"] > 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["value"] == d["value"]
    assert d["e2e"] == {"value": d["value"], "unit": "ms", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    assert d["config"]["workload"] == workload and d["gpu_launches"] == 0
