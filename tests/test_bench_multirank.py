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
