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


def test_default_line_is_the_largest_fp64_config_and_per_config_covers_the_rest():
    """the driver runs the default, so the default must be configs[2] (N = 8192) and carry every other
    BASELINE.json config as a per_config record."""
    sys.path.insert(0, ROOT)
    import bench
    from paper_2401_13772_b200 import hamiltonians as hm

    assert bench.DEFAULT_WORKLOAD == "dense_n8192"
    names = [n for n, _ in bench.PER_CONFIG]
    assert names == ["dense_n256", "dense_n2048", "mixed_bf16x3_n16384", "mixed_n16384", "ellpack_n65536",
                     "ellpack_n65536_literal"]
    for n in names:
        cfg = bench.workload_config(n)
        assert cfg["workload"] == n and "model" not in cfg
    assert "BF16 x 3" in bench.workload_config("mixed_bf16x3_n16384")["arithmetic"]
    assert "FP16 x 2" in bench.workload_config("mixed_n16384")["arithmetic"]
    assert hm.WORKLOADS["dense_n8192"].N == 8192


def test_traffic_is_read_from_the_committed_capture_summary(tmp_path, monkeypatch):
    """roofline.traffic comes from profiles/r02_traffic.json, which `bench.py --traffic-from` writes from an
    `ncu --page raw --csv` export (units row under the header row, one row per profiled launch)."""
    import json

    sys.path.insert(0, ROOT)
    import bench

    committed = json.load(open(bench.TRAFFIC_JSON))
    for name in ("dense_n8192", "dense_n2048", "mixed_n16384", "mixed_bf16x3_n16384", "ellpack_n65536"):
        assert committed[name]["dram_bytes_per_launch"] > 0 and committed[name]["source"].startswith("profiles/")
        assert bench.ncu_traffic(name)["bytes"] == committed[name]["dram_bytes_per_launch"]
    assert bench.ncu_traffic("no_such_workload")["bytes"] is None

    csv = tmp_path / "raw.csv"
    csv.write_text(
        '"ID","Kernel Name","dram__bytes_read.sum","dram__bytes_write.sum"\n'
        '"","","Mbyte","Kbyte"\n'
        '"0","k_a(int)","10.5","2,000"\n'
        '"1","k_b<1>(double)","1","0"\n'
        '"2","k_a(int)","11.5","4,000"\n')
    monkeypatch.setattr(bench, "TRAFFIC_JSON", str(tmp_path / "t.json"))
    bench.write_traffic(str(csv), "w", ["k_a", "k_b"], "unit test")
    got = json.load(open(tmp_path / "t.json"))["w"]
    assert got["kernels"]["k_a"] == {"launches": 2, "dram_bytes_read": 11.0e6, "dram_bytes_write": 3.0e6}
    assert got["dram_bytes_per_launch"] == 11.0e6 + 3.0e6 + 1.0e6
    assert bench.ncu_traffic("w")["bytes"] == 15.0e6
