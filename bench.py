#!/usr/bin/env python
"""bench.py -- SP2 time-to-D on one B200 (BASELINE.json metric), roofline of the dominant kernel, CPU-oracle baseline.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload dense_n2048] [--impl ours|reference]

Workloads: the BASELINE.json configs (dense_n256, dense_n2048, dense_n8192 [default], mixed_n16384 (FP16 x 2 split),
mixed_bf16x3_n16384 (the BF16 split BASELINE.json names), ellpack_n65536 (the labelled stand-in 5'), ellpack_n65536_literal);
the default run also measures all the others and attaches them to its JSON line as `per_config` and, for the Chebyshev expansion of PAPER.md IV.B, cheby_n500 / n1000 / n2000 / n4000 / n8000 (one step =
one bml_chebyshev_dense call; metric chebyshev_time_to_D_ms) and, for the graph-based construction of VIII.B,
graph_n1536 / graph_n12800 (one step = one bml_graph_chebyshev_ellpack call; metric graph_time_to_D_ms).

A "step" is one whole pass of the hot path: one bml_sp2_dense (or bml_sp2_ellpack) solve = Gershgorin bounds +
rescale + every fused X^2 product until the stop rule + output copy, on a seeded synthetic Hamiltonian.
Prints ONE JSON line.  The path does not shard (north_star: one GPU, no collectives):
with --gpus N > 1 (torchrun) every rank solves its own replica and the time is the max over ranks.
"""
from __future__ import annotations

import argparse
import json
import math
import os
import statistics
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

METRIC = "sp2_time_to_D_ms"
DEFAULT_WORKLOAD = "dense_n8192"            # BASELINE.json configs[2]: the largest FP64 single-GPU configuration
METRIC_CHEBY = "chebyshev_time_to_D_ms"     # SURVEY 8(f) item f-1 workloads (--workload cheby_n*)
METRIC_GRAPH = "graph_time_to_D_ms"         # SURVEY 8(f) item f-2 workloads (--workload graph_n*, graph_sp2_n*)
PAPER_DSMS = 148 * 64 * 2  # flops per clock of the FP64 tensor pipe: 148 SMs x 64 FMA/clk/SM


# ----------------------------------------------------------------------------------------------------------
# workload description (algorithmic work per product: DESIGN.md "Roofline")
# ----------------------------------------------------------------------------------------------------------
def dense_flops_per_product(N: int) -> float:
    """Executed flops of one symmetric-square product: upper-triangle BT x BT tiles incl. the diagonal tiles,
    2 * BT * BT * N flops each (2 N^3 (1 + 1/T) / 2 when BT | N); BT = 128 above N = 1024."""
    bt = 32 if N <= 512 else (64 if N <= 1024 else 128)      # dense_fp64_tile() of the library
    T = (N + bt - 1) // bt
    return 2.0 * (T * (T + 1) // 2) * float(bt) * float(bt) * N


# dram__bytes_read.sum + dram__bytes_write.sum of ONE launch of the dominant kernel come from the committed ncu captures:
# profiles/r02_traffic.json, written by `python bench.py --traffic-from <ncu raw csv> --workload W` from the
# `ncu -i <rep> --page raw --csv` export of an `ncu --set full` capture (the .md beside it names the capture command).
TRAFFIC_JSON = os.path.join(ROOT, "profiles", "r02_traffic.json")


def ncu_traffic(workload: str):
    """{'bytes': per-launch DRAM bytes of the workload's dominant kernel(s) or None, 'source': where it came from}."""
    try:
        entry = json.load(open(TRAFFIC_JSON)).get(workload)
    except (OSError, ValueError):
        entry = None
    if not entry:
        return {"bytes": None, "source": "no ncu capture of this workload in profiles/r02_traffic.json"}
    return {"bytes": float(entry["dram_bytes_per_launch"]), "source": entry.get("source", "profiles/r02_traffic.json")}


def write_traffic(csv_path: str, workload: str, kernels: list[str], note: str = ""):
    """Parse an `ncu --page raw --csv` export: per kernel name in `kernels` (substring match) the mean per-launch
    dram__bytes_read.sum + dram__bytes_write.sum; their sum is stored as the workload's per-launch traffic."""
    import csv

    rows = list(csv.reader(open(csv_path)))
    hdr = next(i for i, r in enumerate(rows) if "Kernel Name" in r)
    names, units = rows[hdr], rows[hdr + 1]
    col = {n: i for i, n in enumerate(names)}
    scale = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9}

    def val(r, key):
        return float(r[col[key]].replace(",", "")) * scale[units[col[key]]]

    per_kernel = {}
    for k in kernels:
        sel = [r for r in rows[hdr + 2:] if len(r) > col["Kernel Name"] and k in r[col["Kernel Name"]]]
        if not sel:
            raise SystemExit(f"kernel {k!r} not in {csv_path}")
        rd = sum(val(r, "dram__bytes_read.sum") for r in sel) / len(sel)
        wr = sum(val(r, "dram__bytes_write.sum") for r in sel) / len(sel)
        per_kernel[k] = {"launches": len(sel), "dram_bytes_read": rd, "dram_bytes_write": wr}
    data = json.load(open(TRAFFIC_JSON)) if os.path.exists(TRAFFIC_JSON) else {}
    data[workload] = {
        "dram_bytes_per_launch": sum(v["dram_bytes_read"] + v["dram_bytes_write"] for v in per_kernel.values()),
        "kernels": per_kernel, "source": "profiles/" + os.path.basename(csv_path), "note": note,
    }
    with open(TRAFFIC_JSON, "w") as f:
        json.dump(data, f, indent=1, sort_keys=True)
        f.write("\n")
    print(json.dumps(data[workload]))


def peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        return json.load(open(path)), "measured"
    return {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0}, "fallback"


# ----------------------------------------------------------------------------------------------------------
# clocks sampler (NVML), DURING the timed region
# ----------------------------------------------------------------------------------------------------------
class ClockSampler:
    def __init__(self, index: int):
        self.index, self.samples, self.reasons, self._stop = index, [], set(), threading.Event()
        self.max_mhz, self.ok = None, False
        try:
            import pynvml

            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = int(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
            self.ok = True
        except Exception:
            self.ok = False
        self.t = threading.Thread(target=self._run, daemon=True)

    def _run(self):
        nv = self.nv
        names = {
            0x8: "hw_slowdown", 0x40: "hw_thermal_slowdown", 0x20: "sw_thermal_slowdown", 0x4: "sw_power_cap",
            0x80: "hw_power_brake_slowdown", 0x2: "applications_clocks_setting",
        }
        while not self._stop.is_set():
            try:
                self.samples.append(int(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
                try:
                    r = int(nv.nvmlDeviceGetCurrentClocksEventReasons(self.h))
                except Exception:
                    r = int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h))
                for bit, name in names.items():
                    if r & bit:
                        self.reasons.add(name)
            except Exception:
                pass
            time.sleep(0.01)

    def __enter__(self):
        if self.ok:
            self.t.start()
        return self

    def __exit__(self, *a):
        self._stop.set()
        if self.ok:
            self.t.join(timeout=1.0)

    def summary(self):
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": ["unavailable"]}
        return {"sm_mhz": statistics.median(self.samples), "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "samples": len(self.samples)}


# ----------------------------------------------------------------------------------------------------------
# the reference arm / cpu_baseline: the oracle, as it stands, on the host cores
# ----------------------------------------------------------------------------------------------------------
def oracle_time_to_D(wname: str, H, budget_s: float, n_products_full: int | None):
    """Time the CPU oracle on `wname`.  Runs the full solve if it fits `budget_s`, else a bounded sample of the first
    p products and extrapolates linearly in the product count (every product costs the same N^3 loop).
    Returns (ms_time_to_D, sample description, cores)."""
    import oracle
    from paper_2401_13772_b200 import hamiltonians as hm

    w = hm.WORKLOADS[wname]
    cores = oracle.omp_threads()
    if w.kind == "dense" and w.N > 6000:
        # a full oracle product is N^3 multiply-adds (minutes to hours here): time one product of the oracle on the
        # leading 4096 x 4096 principal block of the same Hamiltonian and scale by (N / 4096)^3 x products
        nb = 4096
        Hb = np.ascontiguousarray(H[:nb, :nb])
        lo, hi = oracle.gershgorin_dense(Hb)
        Xb = oracle.rescale_dense(Hb, lo, hi)
        t0 = time.perf_counter()
        oracle.x2_dense(Xb)
        per = (time.perf_counter() - t0) * (w.N / nb) ** 3
        full = n_products_full or 32
        return per * full * 1e3, (f"one oracle product on the leading {nb}x{nb} principal block, "
                                  f"scaled by ({w.N}/{nb})^3 x {full} products"), cores
    if w.kind == "dense":
        t0 = time.perf_counter()
        _, st = oracle.sp2_dense(H, w.n_occ, w.idem_tol, 2)          # 2 products: calibrates the per-product cost
        per = (time.perf_counter() - t0) / 2
        full = n_products_full or 32
        if per * full <= budget_s:
            t0 = time.perf_counter()
            _, st = oracle.sp2_dense(H, w.n_occ, w.idem_tol, 100)
            dt = time.perf_counter() - t0
            return dt * 1e3, f"full oracle solve, {st['n_products']} products", cores
        p = max(1, min(full, int(budget_s / per)))
        t0 = time.perf_counter()
        _, st = oracle.sp2_dense(H, w.n_occ, w.idem_tol, p)
        dt = time.perf_counter() - t0
        return dt / p * full * 1e3, f"first {p} of {full} products timed, scaled by {full}/{p}", cores
    t0 = time.perf_counter()
    _, st = oracle.sp2_ellpack(*H, w.n_occ, w.idem_tol, w.drop_tol, 1)
    per = time.perf_counter() - t0
    full = n_products_full or 12
    p = max(1, min(full, int(budget_s / max(per, 1e-9))))
    t0 = time.perf_counter()
    _, st = oracle.sp2_ellpack(*H, w.n_occ, w.idem_tol, w.drop_tol, p)
    dt = time.perf_counter() - t0
    if p == full:
        return dt * 1e3, f"full oracle solve, {st['n_products']} products", cores
    return dt / p * full * 1e3, f"first {p} of {full} products timed, scaled by {full}/{p}", cores


def oracle_cheby_time_to_D(wname: str, H, budget_s: float):
    """Time the Chebyshev oracle (oracle/chebyshev.py, chebyshev_ps: the same k + m - 2 products as the GPU path, numpy
    FP64) on `wname`; above N = 2500 a bounded sample: two products 2 A B - C and two scaled additions at full size,
    scaled to the k + m - 2 products and k m additions of the expansion.  Also times the LAPACK diagonalisation route
    (what Fig. 3 of the paper divides by) when it fits the budget.  Returns (ms, sample, cores, extra dict)."""
    from oracle import chebyshev as och
    from paper_2401_13772_b200 import hamiltonians as hm

    w = hm.WORKLOADS[wname]
    try:
        from threadpoolctl import threadpool_info

        cores = max([int(t.get("num_threads", 1)) for t in threadpool_info()] or [1])      # the BLAS pool numpy uses
    except Exception:
        cores = os.cpu_count() or 1
    extra = {}
    if w.N <= 2500:
        t0 = time.perf_counter()
        och.chebyshev_ps(H, w.mu, w.beta, w.k, w.m)
        ms = (time.perf_counter() - t0) * 1e3
        sample = f"full oracle expansion (chebyshev_ps), {w.k + w.m - 2} products, numpy/BLAS threads"
    else:
        emin, emax = och.gershgorin(H)
        Ht = och.map_to_unit(H, emin, emax)
        t0 = time.perf_counter()
        T2 = och.symm_ab(Ht, Ht, None, 2.0, 0.0, -1.0)
        och.symm_ab(T2, Ht, Ht, 2.0, -1.0, 0.0)
        per = (time.perf_counter() - t0) / 2
        t0 = time.perf_counter()
        S = 0.3 * Ht
        S = S + 0.2 * T2
        axpy = (time.perf_counter() - t0) / 2
        ms = (per * (w.k + w.m - 2) + axpy * w.k * w.m) * 1e3
        sample = (f"2 of {w.k + w.m - 2} oracle products and 2 of {w.k * w.m} scaled additions timed at full size, "
                  "scaled; the oracle's products are numpy matmul (BLAS threads), not plain loops")
    if w.N <= 4000 and budget_s >= 20.0:
        t0 = time.perf_counter()
        och.fermi_exact(H, w.mu, w.beta)
        extra["diagonalisation_ms"] = (time.perf_counter() - t0) * 1e3
        extra["diagonalisation_note"] = "numpy.linalg.eigh + U f(Lambda) U^T on the host: the route Fig. 3 compares with"
    return ms, sample, cores, extra


def oracle_graph_time_to_D(wname: str, H):
    """Time the graph oracle (oracle/graph.py) on `wname`: halo lists and gathers of every part as they stand (Python
    loops), the local Fermi operators as a bounded sample -- two steps of the plain recursion Eq. 9 at the size of the
    first part, scaled to the L - 1 products of every part (the oracle's parity target is the plain series).
    Returns (ms, sample, cores)."""
    from oracle import chebyshev as och
    from oracle import graph as og
    from paper_2401_13772_b200 import hamiltonians as hm

    w = hm.WORKLOADS[wname]
    try:
        from threadpoolctl import threadpool_info

        cores = max([int(t.get("num_threads", 1)) for t in threadpool_info()] or [1])
    except Exception:
        cores = os.cpu_count() or 1
    offs, nodes = og.regular_partition(w.N, w.n_parts)
    t0 = time.perf_counter()
    parts = [og.core_halo(*H, nodes[offs[p]: offs[p + 1]], w.graph_tol) for p in range(w.n_parts)]
    subs = [og.matrix2submatrix(*H, pn) for pn, _ in parts]
    t_move = time.perf_counter() - t0
    h = subs[0]
    emin, emax = och.gershgorin(h)
    Ht = och.map_to_unit(h, emin, emax)
    t0 = time.perf_counter()
    T2 = 2.0 * (Ht @ Ht) - np.eye(h.shape[0])
    T3 = 2.0 * (Ht @ T2) - Ht
    per = (time.perf_counter() - t0) / 2
    L = w.k * w.m - 1
    scale = sum((sub.shape[0] / h.shape[0]) ** 3 for sub in subs)
    ms = (t_move + per * (L - 1) * scale) * 1e3
    return ms, (f"halo lists + gathers of all {w.n_parts} parts timed in full ({t_move:.1f} s); 2 of {L - 1} recursion "
                f"products timed at part size {h.shape[0]}, scaled to all parts; products are numpy matmul (BLAS threads), "
                "not plain loops"), cores


def oracle_graph_sp2_time_to_D(wname: str, H, n_products):
    """Time the graph-SP2 oracle (oracle/graph.py graph_sp2) on `wname` as a bounded sample: the halo lists and gathers of
    every part in full (Python loops), and ONE plain triple-loop product (oracle.x2_dense) on the leading 2048 x 2048
    block of the first part, scaled by sum_p (n_p / 2048)^3 x products (every product of the oracle is that loop).
    Returns (ms, sample, cores)."""
    import oracle
    from oracle import graph as og
    from paper_2401_13772_b200 import hamiltonians as hm

    w = hm.WORKLOADS[wname]
    offs, nodes = og.regular_partition(w.N, w.n_parts)
    t0 = time.perf_counter()
    parts = [og.core_halo(*H, nodes[offs[p]: offs[p + 1]], w.graph_tol) for p in range(w.n_parts)]
    subs = [og.matrix2submatrix(*H, pn) for pn, _ in parts]
    t_move = time.perf_counter() - t0
    nb = min(2048, subs[0].shape[0])
    lo, hi = oracle.gershgorin_ellpack(*H)
    Xb = oracle.rescale_dense(np.ascontiguousarray(subs[0][:nb, :nb]), lo, hi)
    t0 = time.perf_counter()
    oracle.x2_dense(Xb)
    per = time.perf_counter() - t0
    full = n_products or 24
    scale = sum((sub.shape[0] / nb) ** 3 for sub in subs)
    ms = (t_move + per * scale * full) * 1e3
    return ms, (f"halo lists + gathers of all {w.n_parts} parts timed in full ({t_move:.1f} s); one oracle product on the "
                f"leading {nb}x{nb} block, scaled by sum_p (n_p/{nb})^3 x {full} products"), oracle.omp_threads()


EXPECTED_PRODUCTS = {"dense_n256": 15, "dense_n2048": 19, "dense_n8192": 32, "mixed_n16384": 30,
                     "mixed_bf16x3_n16384": 30, "ellpack_n65536": 12}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    from paper_2401_13772_b200 import hamiltonians as hm

    w = hm.WORKLOADS[args.workload]
    if w.kind == "ellblock":
        H = hm.make_ellblock(args.workload)
    else:
        H = hm.make_dense(args.workload) if w.kind in ("dense", "cheby") else hm.make_ellpack(args.workload)
    total = args.steps + args.warmup
    budget = max(1.0, 200.0 / total)       # whole run within a few minutes
    times, sample, cores = [], "", 1
    for it in range(total):
        if w.kind == "cheby":
            ms, sample, cores, _ = oracle_cheby_time_to_D(args.workload, H, 0.0)
        elif w.kind == "graph":
            ms, sample, cores = oracle_graph_time_to_D(args.workload, H)
        elif w.kind == "graph_sp2":
            ms, sample, cores = oracle_graph_sp2_time_to_D(args.workload, H, None)
        elif w.kind == "ellblock":
            import oracle

            lo, hi = oracle.gershgorin_ellblock(*H)
            X0 = oracle.rescale_ellblock(*H, lo, hi)[:3]
            t0 = time.perf_counter()
            oracle.x2_ellblock(*X0, w.drop_tol)
            ms = (time.perf_counter() - t0) * 12 * 1e3
            sample, cores = "one oracle block product on X_0 timed, x 12 products", oracle.omp_threads()
        else:
            ms, sample, cores = oracle_time_to_D(args.workload, H, budget, EXPECTED_PRODUCTS.get(args.workload))
        if it >= args.warmup:
            times.append(ms)
    v = float(np.mean(times))
    line = {
        "impl": "reference", "metric": {"cheby": METRIC_CHEBY, "graph": METRIC_GRAPH, "graph_sp2": METRIC_GRAPH}.get(w.kind, METRIC), "value": v, "unit": "ms", "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": v, "higher_is_better": False, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": workload_config(args.workload),
        "cpu_baseline": {"value": v, "unit": "ms", "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": v, "unit": "ms", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)
    return 0


def workload_config(name: str):
    from paper_2401_13772_b200 import hamiltonians as hm

    w = hm.WORKLOADS[name]
    cfg = {"workload": name, "kind": w.kind, "N": w.N, "n_occ": w.n_occ, "idem_tol": w.idem_tol, "note": w.note,
           "seed": 0, "max_products": 100,
           "l2": "flushed between steps (256 MiB write > the 126 MB L2)"}
    if w.kind == "dense":
        resident = 3 * w.N * w.N * 8 / 2**20
        cfg["l2"] += (f"; H + both iterates are {resident:.0f} MiB: " +
                      ("they then stay L2-resident within a step, which is part of the method" if resident < 120
                       else "larger than L2, every product streams its operands from HBM"))
        cfg["arithmetic"] = {0: "fp64 (DMMA)", 1: "mixed: FP16 x 2 split products on tcgen05, FP64 elsewhere "
                                "(NOT the split BASELINE.json names; see mixed_bf16x3_n16384)",
                             2: "mixed: BF16 x 3 split products on tcgen05, FP64 elsewhere (the BF16 split of "
                                "BASELINE.json configs[3])"}[w.precision]
    if w.kind == "ellpack":
        cfg.update({"M": w.M, "drop_tol": w.drop_tol})
    if w.kind == "ellblock":
        cfg["l2"] = "flushed between steps (256 MiB write)"
        cfg.update({"bs": w.bs, "MB": w.MB, "drop_tol": w.drop_tol, "drop_rule": "block Frobenius norm >= drop_tol or diagonal block"})
    if w.kind == "graph_sp2":
        cfg["l2"] = "flushed between steps (256 MiB write)"
        cfg.update({"M": w.M, "M_out": w.M_out, "n_parts": w.n_parts, "graph_tol": w.graph_tol, "drop_tol": w.drop_tol,
                    "partition": "regular index segments", "local_solver": "SP2, one polynomial for all parts"})
    if w.kind == "graph":
        for key in ("n_occ", "idem_tol", "max_products"):
            cfg.pop(key)
        cfg["l2"] = "flushed between steps (256 MiB write)"
        cfg.update({"M": w.M, "M_out": w.M_out, "n_parts": w.n_parts, "graph_tol": w.graph_tol, "drop_tol": w.drop_tol,
                    "mu": w.mu, "beta": w.beta, "k": w.k, "m": w.m, "L": w.k * w.m - 1,
                    "partition": "regular index segments"})
    if w.kind == "cheby":
        for key in ("n_occ", "idem_tol", "max_products"):
            cfg.pop(key)
        cfg["l2"] = "flushed between steps (256 MiB write)"
        cfg.update({"mu": w.mu, "beta": w.beta, "k": w.k, "m": w.m, "L": w.k * w.m - 1,
                    "products": w.k + w.m - 2})
    return cfg


# ----------------------------------------------------------------------------------------------------------
# multi-rank aggregation (replicas only: DESIGN.md 7)
# ----------------------------------------------------------------------------------------------------------
def aggregate_over_ranks(values, dist=None, device=None):
    """MAX over ranks of each timing in `values` (the slowest replica sets the job time).  `dist` is an initialised
    torch.distributed module or None for a single process.  No data-path collective exists: this is the only one."""
    import torch

    if dist is None:
        return [float(v) for v in values]
    t = torch.tensor(list(values), dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(v) for v in t.tolist()]


def replicas_per_second(world: int, ms: float) -> float:
    """Whole-job throughput of `world` independent replicas that each finish one solve in <= ms."""
    return world / (ms * 1e-3)


# ----------------------------------------------------------------------------------------------------------
# scaffolding shared by the three arms (SP2, Chebyshev, graph): process setup, the timed loop, a kernel timed alone
# ----------------------------------------------------------------------------------------------------------
class Ranks:
    """One process per GPU (torchrun env), NCCL only for the barrier and the max-over-ranks of the timings."""

    def __init__(self):
        import torch

        self.world = int(os.environ.get("WORLD_SIZE", "1"))
        self.rank = int(os.environ.get("RANK", "0"))
        self.local = int(os.environ.get("LOCAL_RANK", "0"))
        if not torch.cuda.is_available():
            raise RuntimeError("bench.py needs a CUDA device: libbmlsp2 has no CPU path")
        torch.cuda.set_device(self.local)
        self.dist = None
        if self.world > 1:
            import torch.distributed as dist

            dist.init_process_group("nccl")
            self.dist = dist
        self.dev = torch.device("cuda", self.local)

    def barrier(self):
        import torch

        if self.dist is not None:
            self.dist.barrier()
        torch.cuda.synchronize()

    def finish(self):
        if self.dist is not None:
            self.dist.destroy_process_group()


def timed_steps(rk: Ranks, solve, args):
    """W untimed warm-up steps, then exactly K steps, each between CUDA events on the launch stream, L2 flushed before
    each, barrier + synchronize on both sides, clocks sampled during the timed region.
    Returns (per-step ms, wall seconds of the timed region, clocks summary, result of the last step)."""
    import torch

    flush = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device=rk.dev)
    res = None
    for _ in range(args.warmup):
        _, res = solve()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    rk.barrier()
    with ClockSampler(rk.local) as clk:
        t0 = time.perf_counter()
        for k in range(args.steps):
            flush.fill_(k & 0xFF)                     # L2 flush, outside the per-step events
            ev[k][0].record()
            _, res = solve()                          # synchronises the stream once, at its end (reads the stats)
            ev[k][1].record()
        rk.barrier()
        t_wall = time.perf_counter() - t0
    return [a.elapsed_time(b) for a, b in ev], t_wall, clk.summary(), res


def time_alone(fn, reps: int, warm: int = 3) -> float:
    """ms per call of `fn` issued back to back on the current stream, after `warm` untimed calls."""
    import torch

    for _ in range(warm):
        fn()
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    a.record()
    for _ in range(reps):
        fn()
    b.record()
    torch.cuda.synchronize()
    return a.elapsed_time(b) / reps


def timed_e2e(rk: Ranks, step, n: int) -> float:
    """ms per end-to-end step (`step` copies the inputs in from pinned host memory, solves, copies the result out and
    synchronises), wall clock, after two untimed steps."""
    for _ in range(2):
        step()
    rk.barrier()
    t0 = time.perf_counter()
    for _ in range(n):
        step()
    return (time.perf_counter() - t0) / n * 1e3


# ----------------------------------------------------------------------------------------------------------
# our arm
# ----------------------------------------------------------------------------------------------------------
def sp2_measure(rk: Ranks, wname: str, steps: int, warmup: int, lanczos_steps: int = 0, e2e_steps: int | None = None):
    """One SP2 workload through the C ABI: W warm-ups + K timed solves on a resident H (CUDA events, L2 flushed between
    steps, clocks sampled), the end-to-end leg with host buffers, and the dominant kernel timed alone against its
    roofline.  Returns (record dict, H as numpy) -- the record is the body of the JSON line / of a per_config entry."""
    import contextlib
    import types

    import torch

    from paper_2401_13772_b200 import api, hamiltonians as hm

    args = types.SimpleNamespace(steps=steps, warmup=warmup)
    dev = rk.dev
    w = hm.WORKLOADS[wname]
    dense = w.kind == "dense"
    sp2_flags = api.FLAG_LANCZOS_BOUNDS(lanczos_steps) if lanczos_steps else 0

    # ---- inputs: seeded synthetic Hamiltonian, resident in HBM; pinned host copies for the e2e leg
    if dense:
        H_np = hm.make_dense(wname)
        H_host = torch.from_numpy(H_np).pin_memory()
        H_dev = H_host.to(dev)
        solver = api.DenseSolver(w.N, dev, precision=w.precision)
        D_host = torch.empty((w.N, w.N), dtype=torch.float64).pin_memory()

        def solve(Hd):
            return solver.solve(Hd, w.n_occ, w.idem_tol, 100, flags=sp2_flags)
    else:
        H_np = hm.make_ellpack(wname)
        H_host = tuple(torch.from_numpy(a).pin_memory() for a in H_np)
        H_dev = tuple(a.to(dev) for a in H_host)
        solver = api.EllpackSolver(w.N, w.M, dev)
        D_host = tuple(torch.empty_like(a).pin_memory() for a in H_host)

        def solve(Hd):
            return solver.solve(*Hd, w.n_occ, w.idem_tol, w.drop_tol, 100, flags=sp2_flags)

    # Small dense matrices run on a stream of their own: the library replays the static head of such a solve as a CUDA
    # graph, which the legacy default stream cannot capture.  Everything else stays on the current stream.
    side = torch.cuda.Stream(dev) if (dense and w.N <= 1024) else None
    if side is not None:
        side.wait_stream(torch.cuda.current_stream())
    with (torch.cuda.stream(side) if side is not None else contextlib.nullcontext()):
        # ---- device-resident timing: W warm-ups, then exactly K timed steps
        step_ms, t_wall, clocks, res = timed_steps(rk, lambda: solve(H_dev), args)
        ms = float(np.mean(step_ms))

        # ---- e2e: host buffers through the public API; H2D of H and D2H of D inside the timed region
        H_in = torch.empty_like(H_dev) if dense else None

        def e2e_step():
            if dense:
                H_in.copy_(H_host, non_blocking=True)
                D, _ = solve(H_in)
                D_host.copy_(D, non_blocking=True)
            else:
                D, _ = solve(tuple(a.to(dev, non_blocking=True) for a in H_host))
                for dst, src in zip(D_host, D):
                    dst.copy_(src, non_blocking=True)
            torch.cuda.synchronize()

        if e2e_steps is None:
            e2e_steps = max(3, min(steps, 10))
        h2d = H_host.numel() * 8 if dense else sum(a.numel() * a.element_size() for a in H_host)
        d2h = h2d
        e2e_ms = timed_e2e(rk, e2e_step, e2e_steps) if res.status >= 0 else float("nan")
    if side is not None:
        torch.cuda.current_stream().wait_stream(side)

    # ---- dominant kernel, timed alone with CUDA events on the launching stream
    pk, pk_src = peaks()
    traffic = ncu_traffic(wname)
    roof = None
    n_prod = int(res.n_products)
    if res.status < 0:
        roof = None
    elif dense and w.precision == 0:
        lo_hi = api.bml_gershgorin(H_dev).cpu().numpy()
        s = 1.0 / (lo_hi[1] - lo_hi[0])
        X0 = api.padded_dense((lo_hi[1] * torch.eye(w.N, dtype=torch.float64) - H_host) * s, dev)
        Xn = torch.empty_strided(X0.shape, X0.stride(), dtype=X0.dtype, device=dev)
        ws = api._workspace(api.load().bml_x2_dense_workspace_bytes(w.N, 0), dev)
        k_ms = time_alone(lambda: api.bml_x2_dense(X0, 1, 0, Xn, ws), 20)
        peak_probe = api.bml_probe_fp64_tensor_peak(40000)
        flops = dense_flops_per_product(w.N)
        achieved = flops / (k_ms * 1e-3) / 1e12
        nominal_ratio_peak = pk["bf16_tflops"] * (40.0 / 2250.0)
        roof = {
            "bound": "tensor",
            "kernel": "x2_dense_fp64_sk_kernel" if w.N > 1024 else "x2_dense_fp64_kernel<%d>" % (32 if w.N <= 512 else 64),
            "achieved": achieved, "peak": peak_probe,
            "unit": "TFLOP/s", "frac": achieved / peak_probe, "traffic": traffic["bytes"], "traffic_source": traffic["source"],
            "algorithmic_bytes": 2.0 * w.N * w.N * 8,
            "peak_source": "FP64 DMMA issue peak measured live by bml_probe_fp64_tensor_peak in this run "
                           "(MEASURED_PEAKS.json has no FP64 entry)",
            "peak_alt_bf16_ratio": nominal_ratio_peak,
            "frac_alt": achieved / nominal_ratio_peak,
            "peak_alt_source": f"{pk_src} bf16 burst x nominal FP64/bf16 ratio 40/2250",
            "launch_ms": k_ms, "flops_per_launch": flops,
            "in_step_tflops": flops * n_prod / (ms * 1e-3) / 1e12,
        }
        del X0, Xn, ws
    elif dense and w.precision != 0:
        # mixed mode: the fused split-plane tcgen05 product, timed alone through bml_x2_dense(precision); that entry
        # point also runs the (HBM-bound, ~2% of the time) FP64 -> 16-bit planes split of its input
        terms = 3.0 if w.precision == 1 else 6.0          # FP16 x 2: hh, hl, lh; BF16 x 3: six cross terms
        lo_hi = api.bml_gershgorin(H_dev).cpu().numpy()
        s = 1.0 / (lo_hi[1] - lo_hi[0])
        X0 = api.padded_dense((lo_hi[1] * torch.eye(w.N, dtype=torch.float64) - H_host) * s, dev)
        Xn = torch.empty_strided(X0.shape, X0.stride(), dtype=X0.dtype, device=dev)
        ws = api._workspace(api.load().bml_x2_dense_workspace_bytes(w.N, w.precision), dev)
        k_ms = time_alone(lambda: api.bml_x2_dense(X0, 1, w.precision, Xn, ws), 10)
        flops = terms * dense_flops_per_product(w.N)      # executed 16-bit tensor flops per product
        achieved = flops / (k_ms * 1e-3) / 1e12
        roof = {
            "bound": "tensor", "kernel": "x2_dense_mixed_kernel", "achieved": achieved, "peak": pk["bf16_tflops"],
            "unit": "TFLOP/s", "frac": achieved / pk["bf16_tflops"], "traffic": traffic["bytes"],
            "traffic_source": traffic["source"],
            "peak_source": f"{pk_src} bf16 burst (cuBLAS) from MEASURED_PEAKS.json (fp16 and bf16 share the tcgen05 "
                           "kind::f16 rate); kernel timed alone (launch includes the FP64 -> 16-bit planes split)",
            "cross_terms": terms,
            "launch_ms": k_ms, "flops_per_launch": flops,
            "in_step_tflops": flops * n_prod / (ms * 1e-3) / 1e12,
            "in_step_frac_of_sustained": flops * n_prod / (ms * 1e-3) / 1e12 / pk["bf16_tflops_sustained"],
            "fp64_equivalent_tflops": dense_flops_per_product(w.N) / (k_ms * 1e-3) / 1e12,
        }
        del X0, Xn, ws
    elif not dense:
        # a mid-sequence iterate: X_5 (the solve stopped after 6 products returns D = X_5)
        Xmid, _ = solver.solve(*H_dev, w.n_occ, w.idem_tol, w.drop_tol, 6)
        Xmid = tuple(t.clone() for t in Xmid)
        nn = Xmid[2].to(torch.int64)
        mask = torch.arange(w.M, device=dev).unsqueeze(0) < nn.unsqueeze(1)
        macs = int((nn[Xmid[1].to(torch.int64)] * mask).sum().item())     # sum_i sum_{k in row i} n_k
        out = tuple(torch.zeros_like(t) for t in Xmid)
        ws = api._workspace(api.load().bml_x2_ellpack_workspace_bytes(w.N, w.M), dev)
        k_ms = time_alone(lambda: api.bml_x2_ellpack(Xmid, 1, w.drop_tol, out, ws), 5, warm=2)
        comp_bytes = float((12 * nn + 4).sum().item() + (12 * out[2].to(torch.int64) + 4).sum().item())
        gathered = 12.0 * macs
        achieved = comp_bytes / (k_ms * 1e-3) / 1e9
        roof = {
            "bound": "hbm", "kernel": "ell_block_summary_kernel + x2_ellpack_upper_kernel (pre-screened small tables, then "
                                      "large tables for the rows passed on) + x2_ellpack_assemble_kernel", "achieved": achieved,
            "peak": pk["hbm_gbs"], "unit": "GB/s", "frac": achieved / pk["hbm_gbs"],
            "frac_uses": "compulsory bytes (read X_5 + write X_6: 12 B per stored entry + 4 B per row)",
            "traffic": traffic["bytes"], "traffic_source": traffic["source"],
            "peak_source": f"{pk_src} copy bandwidth from MEASURED_PEAKS.json",
            "note": "SURVEY 8(d): three byte counts.  `frac` uses the COMPULSORY bytes; the kernel is bound by "
                    "shared-memory hash updates and issue slots, not HBM (DESIGN.md 5.4), so that fraction is small by "
                    "construction; the gathered-bytes rate is what BASELINE.json's '>= 60% of HBM' can be read on",
            "launch_ms": k_ms,
            "bytes": {
                "compulsory": {"bytes": comp_bytes, "gbs": achieved, "frac_of_hbm": achieved / pk["hbm_gbs"]},
                "ncu_dram": None if traffic["bytes"] is None else {
                    "bytes": traffic["bytes"], "gbs": traffic["bytes"] / (k_ms * 1e-3) / 1e9,
                    "frac_of_hbm": traffic["bytes"] / (k_ms * 1e-3) / 1e9 / pk["hbm_gbs"]},
                "gathered": {"bytes": gathered, "gbs": gathered / (k_ms * 1e-3) / 1e9,
                             "frac_of_hbm": gathered / (k_ms * 1e-3) / 1e9 / pk["hbm_gbs"]},
            },
            "compulsory_bytes": comp_bytes, "macs_per_launch": macs,
            "macs_note": "full-row Gustavson count sum_i sum_{k in i} n_k; the kernel executes about half of them "
                         "(columns j >= i only, mirrored by symmetry)",
            "gathered_gbs": gathered / (k_ms * 1e-3) / 1e9, "gmacs_per_s": macs / (k_ms * 1e-3) / 1e9,
            "mean_row_nnz": float(nn.double().mean().item()),
        }
        del Xmid, out, ws

    # product launches of one solve: a first batch of 16, then batches of 8 kept one batch ahead of the device until
    # the host sees the stop flag (api.cu enqueue_products); launches behind the stop flag exit at once on the device
    n_enq = 16
    while n_enq < 100:
        n_enq += 8
        if n_enq - 8 >= max(n_prod, 16):
            break
    n_enq = min(n_enq, 100)
    pre = (2 + 1 + 1 + 1 + (1 if w.precision != 0 else 0)) if dense else (2 + 2 + 1)
    # a mixed product is the FP64-diagonal kernel + the tcgen05 kernel; a sparse product is the column-block summary, the
    # pre-screened small-table kernel, the large-table kernel for the rows it passed on, and the assemble kernel (two
    # kernels when the pre-screen does not apply: tau = 0, M > 512 or N > 131072)
    ell_screened = (not dense) and w.drop_tol > 0 and w.M <= 512 and w.N <= 131072
    per_product = 1 if (dense and w.precision == 0) else (2 if dense else (4 if ell_screened else 2))
    launches_per_step = pre + n_enq * per_product + 1
    if dense and w.precision == 0 and w.N <= 1024:
        launches_per_step = pre + 1 + 1           # all products run inside ONE cooperative launch (whole-solve kernel)
    rec = {
        "ms": ms, "step_ms": step_ms, "t_wall": t_wall, "clocks": clocks, "res": res, "n_products": n_prod,
        "e2e_ms": e2e_ms, "e2e_steps": e2e_steps, "h2d": int(h2d), "d2h": int(d2h), "roofline": roof,
        "launches_per_step": launches_per_step,
        "dtype": {0: "f64", 1: "fp16x2 split products (fp32 TMEM chunks) + f64 accumulate/update",
                  2: "bf16x3 split products (fp32 TMEM chunks) + f64 accumulate/update"}[w.precision if dense else 0],
    }
    del solver, H_dev, H_host, D_host
    torch.cuda.empty_cache()
    return rec, H_np


# the other BASELINE.json configs, measured in the same run and attached to the default line as `per_config`
PER_CONFIG = [("dense_n256", 10), ("dense_n2048", 10), ("mixed_bf16x3_n16384", 3), ("mixed_n16384", 3),
              ("ellpack_n65536", 3), ("ellpack_n65536_literal", 1)]


def per_config_block(rk: Ranks, skip: str, only=None):
    out = {}
    for wname, steps in PER_CONFIG:
        if wname == skip or (only and wname not in only):
            continue
        t0 = time.perf_counter()
        try:
            rec, _ = sp2_measure(rk, wname, steps, 3, 0, e2e_steps=2)
        except Exception as e:      # one config must not take the headline down with it
            out[wname] = {"error": f"{type(e).__name__}: {e}"}
            continue
        res = rec["res"]
        out[wname] = {
            "config": workload_config(wname), "dtype": rec["dtype"], "ms": rec["ms"], "steps": steps, "warmup": 3,
            "step_ms_min": float(min(rec["step_ms"])), "step_ms_max": float(max(rec["step_ms"])),
            "status": int(res.status), "status_string": res.message, "n_products": rec["n_products"],
            "branch": res.branch, "max_row_nnz": [int(x) for x in res.max_row_nnz] if "ellpack" in wname else None,
            "overflow_row": int(res.overflow_row),
            "e2e": {"value": rec["e2e_ms"], "unit": "ms", "h2d_bytes_per_step": rec["h2d"],
                    "d2h_bytes_per_step": rec["d2h"], "steps": rec["e2e_steps"]},
            "roofline": rec["roofline"], "clocks": rec["clocks"], "gpu_launches_per_step": rec["launches_per_step"],
            "bench_wall_s": round(time.perf_counter() - t0, 1),
        }
    # the widening rows of SURVEY 8(f) (not BASELINE.json configs), so that their numbers are in the driver-run record
    # too: the Chebyshev expansion (f-1), the graph-based construction with SP2 as the local solver (f-2), SP2 from
    # Lanczos-tightened bounds (f-3) and the ELLBLOCK path (f-4)
    if not (only and "dense_n8192_lanczos32" not in only):
        t0 = time.perf_counter()
        try:
            rec, _ = sp2_measure(rk, "dense_n8192", 3, 3, 32, e2e_steps=2)
            res = rec["res"]
            out["dense_n8192_lanczos32"] = {
                "config": workload_config("dense_n8192"), "row": "SURVEY 8(f) f-3", "dtype": rec["dtype"], "ms": rec["ms"],
                "steps": 3, "warmup": 3, "status": int(res.status), "n_products": rec["n_products"], "branch": res.branch,
                "spectral_bounds": {"emin": res.emin, "emax": res.emax, "kind": "lanczos(32) within gershgorin"},
                "e2e": {"value": rec["e2e_ms"], "unit": "ms", "h2d_bytes_per_step": rec["h2d"],
                        "d2h_bytes_per_step": rec["d2h"], "steps": rec["e2e_steps"]},
                "roofline": rec["roofline"], "clocks": rec["clocks"], "bench_wall_s": round(time.perf_counter() - t0, 1),
            }
        except Exception as e:
            out["dense_n8192_lanczos32"] = {"error": f"{type(e).__name__}: {e}"}
    for wname, fn, tag in (("cheby_n2000", run_cheby, "SURVEY 8(f) f-1"), ("graph_sp2_n12800", run_graph_sp2, "SURVEY 8(f) f-2"),
                           ("ellblock_n65536", run_ellblock, "SURVEY 8(f) f-4")):
        if wname == skip or (only and wname not in only):
            continue
        t0 = time.perf_counter()
        try:
            sub = argparse.Namespace(workload=wname, steps=3, warmup=3, no_cpu_baseline=True)
            rec = fn(sub, rk=rk, emit=False)
        except Exception as e:
            out[wname] = {"error": f"{type(e).__name__}: {e}"}
            continue
        rec = {k: rec[k] for k in ("config", "dtype", "value", "steps", "warmup", "step_ms_min", "step_ms_max", "status",
                                   "n_products", "branch", "ms_per_product", "e2e", "roofline", "clocks") if k in rec}
        rec["ms"] = rec.pop("value")
        rec["row"] = tag
        rec["bench_wall_s"] = round(time.perf_counter() - t0, 1)
        out[wname] = rec
    return out


def run_ours(args):
    from paper_2401_13772_b200 import api

    rk = Ranks()
    api.load()
    dev, dist, world, rank = rk.dev, rk.dist, rk.world, rk.rank
    rec, H_np = sp2_measure(rk, args.workload, args.steps, args.warmup, args.lanczos_steps)
    res, n_prod, step_ms, clocks = rec["res"], rec["n_products"], rec["step_ms"], rec["clocks"]
    launches_per_step = rec["launches_per_step"]

    # ---- aggregate over ranks: max time
    ms, e2e_ms = aggregate_over_ranks([rec["ms"], rec["e2e_ms"]], dist, dev)

    if rank != 0:
        rk.finish()
        return 0

    # ---- the other configs of BASELINE.json (one GPU, default run only)
    per_config = None
    if world == 1 and args.per_config:
        per_config = per_config_block(rk, args.workload, [x for x in args.per_config_list.split(",") if x])

    # ---- CPU oracle baseline (rank 0, N = 1 only): bounded sample, ~10-30 s
    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        v, sample, cores = oracle_time_to_D(args.workload, H_np, 25.0, n_prod)
        cpu = {"value": v, "unit": "ms", "cores": cores, "kind": "oracle", "sample": sample}

    line = {
        "metric": METRIC, "value": ms, "unit": "ms", "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms, "higher_is_better": False, "scaling": "weak", "vs_baseline": None,
        "dtype": rec["dtype"],
        "data": "synthetic", "config": workload_config(args.workload),
        "status": int(res.status), "n_products": n_prod, "branch": res.branch,
        "spectral_bounds": {"emin": res.emin, "emax": res.emax,
                            "kind": f"lanczos({args.lanczos_steps}) within gershgorin" if args.lanczos_steps else "gershgorin"},
        "step_ms_min": float(min(step_ms)), "step_ms_max": float(max(step_ms)), "wall_s_timed_region": rec["t_wall"],
        "ms_per_product": ms / max(n_prod, 1),
        "aggregate_solves_per_s": replicas_per_second(world, ms),
        "e2e": {"value": e2e_ms, "unit": "ms", "h2d_bytes_per_step": rec["h2d"], "d2h_bytes_per_step": rec["d2h"],
                "steps": rec["e2e_steps"]},
        "gpu_launches": launches_per_step * args.steps,
        "gpu_launches_note": f"{launches_per_step} per step (upper bound: the host stops enqueueing one or two batches of "
                             f"8 after the stop flag); {n_prod} product launches do work, the rest exit on the "
                             "device-side stop flag",
        "roofline": rec["roofline"], "cpu_baseline": cpu, "clocks": clocks, "per_config": per_config,
    }
    print(json.dumps(line), flush=True)
    rk.finish()
    return 0


# ----------------------------------------------------------------------------------------------------------
# our arm, Chebyshev workloads: same contract, one bml_chebyshev_dense call per step
# ----------------------------------------------------------------------------------------------------------
def run_cheby(args, rk=None, emit=True):
    """emit=False: return the JSON record instead of printing it (per_config of the default run; `rk` is the caller's)."""
    import torch

    from paper_2401_13772_b200 import api, hamiltonians as hm

    rk = rk or Ranks()
    api.load()
    dev = rk.dev
    w = hm.WORKLOADS[args.workload]
    H_np = hm.make_dense(args.workload)
    H_host = torch.from_numpy(H_np).pin_memory()
    H_dev = H_host.to(dev)
    solver = api.ChebyshevSolver(w.N, w.k, w.m, dev)
    D_host = torch.empty((w.N, w.N), dtype=torch.float64).pin_memory()

    # a stream of its own: the library replays small expansions as a CUDA graph, which the legacy default stream
    # cannot capture (the events of timed_steps are recorded on the current stream, i.e. this one)
    side = torch.cuda.Stream(dev)
    side.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(side):
        step_ms, t_wall, clocks, res = timed_steps(rk, lambda: solver.solve(H_dev, w.mu, w.beta), args)
        ms = float(np.mean(step_ms))

        H_in = torch.empty_like(H_dev)

        def e2e_step():
            H_in.copy_(H_host, non_blocking=True)
            D, _ = solver.solve(H_in, w.mu, w.beta)
            D_host.copy_(D, non_blocking=True)
            torch.cuda.synchronize()

        e2e_steps = max(3, min(args.steps, 10))
        h2d = d2h = H_host.numel() * 8
        e2e_ms = timed_e2e(rk, e2e_step, e2e_steps)
    torch.cuda.current_stream().wait_stream(side)

    # dominant kernel: one product alpha A B + beta C + gamma I of this size, timed alone
    T1 = (2.0 * H_host - (res.emax + res.emin) * torch.eye(w.N, dtype=torch.float64)) / (res.emax - res.emin)
    slab, n, ld, _ = api.matrix_slab([T1, T1 @ T1, torch.zeros_like(T1)], dev)
    ws = api._workspace(api.load().bml_symm_ab_workspace_bytes(), dev)
    job = [(0, 1, 0, 2, 2.0, -1.0, 0.0)]
    k_ms = time_alone(lambda: api.bml_symm_ab_dense(slab, n, ld, job, ws), 20)
    peak_probe = api.bml_probe_fp64_tensor_peak(40000)
    flops = dense_flops_per_product(w.N)
    achieved = flops / (k_ms * 1e-3) / 1e12
    n_prod = int(res.n_products)
    bt = 32 if w.N <= 512 else (64 if w.N <= 1024 else 128)
    pk, pk_src = peaks()
    sums_bytes = float(w.k - 1 + w.m) * w.N * w.N * 8
    roof = {
        "bound": "tensor", "kernel": "symm_ab_fp64_kernel<%d>" % bt, "achieved": achieved, "peak": peak_probe,
        "unit": "TFLOP/s", "frac": achieved / peak_probe, "traffic": ncu_traffic(args.workload)["bytes"],
        "peak_source": "FP64 DMMA issue peak measured live by bml_probe_fp64_tensor_peak in this run "
                       "(MEASURED_PEAKS.json has no FP64 entry)",
        "launch_ms": k_ms, "flops_per_launch": flops,
        "in_step_tflops": flops * n_prod / (ms * 1e-3) / 1e12,
        "sums_kernel": {"bound": "hbm", "kernel": "cheb_sums_kernel", "bytes_per_launch": sums_bytes,
                        "ms_at_peak": sums_bytes / (pk["hbm_gbs"] * 1e9) * 1e3, "peak": pk["hbm_gbs"],
                        "peak_source": f"{pk_src} copy bandwidth from MEASURED_PEAKS.json"},
    }
    ms, e2e_ms = aggregate_over_ranks([ms, e2e_ms], rk.dist, dev)
    if rk.rank != 0:
        rk.finish()
        return 0
    cpu = None
    if rk.world == 1 and not args.no_cpu_baseline:
        v, sample, cores, extra = oracle_cheby_time_to_D(args.workload, H_np, 25.0)
        cpu = {"value": v, "unit": "ms", "cores": cores, "kind": "oracle", "sample": sample, **extra}
    # gershgorin (2) + coefficients + map + product launches + partial sums + trace
    launches_per_step = 2 + 1 + 1 + int(res.n_launches) + 1 + 1
    line = {
        "metric": METRIC_CHEBY, "value": ms, "unit": "ms", "n_gpus": rk.world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms, "higher_is_better": False, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic", "config": workload_config(args.workload),
        "status": int(res.status), "n_products": n_prod, "n_product_launches": int(res.n_launches),
        "trace_D": res.trace, "step_ms_min": float(min(step_ms)), "step_ms_max": float(max(step_ms)),
        "wall_s_timed_region": t_wall, "ms_per_product": ms / max(n_prod, 1),
        "aggregate_solves_per_s": replicas_per_second(rk.world, ms),
        "e2e": {"value": e2e_ms, "unit": "ms", "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h),
                "steps": e2e_steps},
        "gpu_launches": launches_per_step * args.steps,
        "gpu_launches_note": f"{launches_per_step} per step: 2 Gershgorin + coefficients + map + "
                             f"{int(res.n_launches)} grouped product launches ({n_prod} products) + partial sums + trace",
        "roofline": roof, "cpu_baseline": cpu, "clocks": clocks,
    }
    if not emit:
        return line
    print(json.dumps(line), flush=True)
    rk.finish()
    return 0


# ----------------------------------------------------------------------------------------------------------
# our arm, graph-based workloads: one bml_graph_chebyshev_ellpack call per step
# ----------------------------------------------------------------------------------------------------------
def run_graph(args):
    import torch

    from paper_2401_13772_b200 import api, hamiltonians as hm

    rk = Ranks()
    api.load()
    dev = rk.dev
    w = hm.WORKLOADS[args.workload]
    H_np = hm.make_ellpack(args.workload)
    H_host = tuple(torch.from_numpy(a).pin_memory() for a in H_np)
    H_dev = tuple(a.to(dev) for a in H_host)
    offs_np, nodes_np = hm.regular_core_partition(w.N, w.n_parts)
    offs, nodes = torch.from_numpy(offs_np).to(dev), torch.from_numpy(nodes_np).to(dev)
    # part sizes are not known before the halo pass: size the workspace from one dry call of the halo kernels
    sizes = api.bml_graph_core_halo(H_dev, offs, nodes, w.graph_tol)[2].cpu().numpy()
    cap = int(sizes[:, 0].max())
    solver = api.GraphSolver(w.N, w.M_out, w.n_parts, cap, w.k, w.m, dev)
    D_host = tuple(torch.empty_like(a).pin_memory() for a in (solver.dv.cpu(), solver.di.cpu(), solver.dn.cpu()))

    def solve(Hd):
        return solver.solve(Hd, offs, nodes, w.graph_tol, w.mu, w.beta, w.drop_tol)

    step_ms, t_wall, clocks, res = timed_steps(rk, lambda: solve(H_dev), args)
    ms = float(np.mean(step_ms))

    def e2e_step():
        D, _ = solve(tuple(a.to(dev, non_blocking=True) for a in H_host))
        for dst, src in zip(D_host, D):
            dst.copy_(src, non_blocking=True)
        torch.cuda.synchronize()

    e2e_steps = max(3, min(args.steps, 10))
    h2d = sum(a.numel() * a.element_size() for a in H_host)
    d2h = sum(a.numel() * a.element_size() for a in D_host)
    e2e_ms = timed_e2e(rk, e2e_step, e2e_steps)

    # dominant kernel: one local-solver product at the size of the largest part, timed alone
    g = torch.Generator().manual_seed(0)
    A = torch.randn((cap, cap), generator=g, dtype=torch.float64) / math.sqrt(cap)
    A = (A + A.T) / 4
    slab, n, ld, _ = api.matrix_slab([A, A, torch.zeros_like(A)], dev)
    ws = api._workspace(api.load().bml_symm_ab_workspace_bytes(), dev)
    job = [(0, 1, 0, 2, 2.0, -1.0, 0.0)]
    k_ms = time_alone(lambda: api.bml_symm_ab_dense(slab, n, ld, job, ws), 10)
    peak_probe = api.bml_probe_fp64_tensor_peak(40000)
    flops = dense_flops_per_product(cap)
    achieved = flops / (k_ms * 1e-3) / 1e12
    n_prod = int(res.n_products)
    step_flops = sum(dense_flops_per_product(int(sz)) for sz in res.part_size) * (w.k + w.m - 2)
    roof = {
        "bound": "tensor", "kernel": "symm_ab_fp64_kernel<128>", "achieved": achieved, "peak": peak_probe,
        "unit": "TFLOP/s", "frac": achieved / peak_probe, "traffic": ncu_traffic(args.workload)["bytes"],
        "peak_source": "FP64 DMMA issue peak measured live by bml_probe_fp64_tensor_peak in this run "
                       "(MEASURED_PEAKS.json has no FP64 entry)",
        "launch_ms": k_ms, "flops_per_launch": flops, "part_size": cap,
        "in_step_tflops": step_flops / (ms * 1e-3) / 1e12,
        "in_step_frac": step_flops / (ms * 1e-3) / 1e12 / peak_probe,
    }
    ms, e2e_ms = aggregate_over_ranks([ms, e2e_ms], rk.dist, dev)
    if rk.rank != 0:
        rk.finish()
        return 0
    cpu = None
    if rk.world == 1 and not args.no_cpu_baseline:
        v, sample, cores = oracle_graph_time_to_D(args.workload, H_np)
        cpu = {"value": v, "unit": "ms", "cores": cores, "kind": "oracle", "sample": sample}
    levels = max(1, math.ceil(math.log2(w.k)))
    # per part: gather, Gershgorin x2, coefficients, map, products, partial sums, trace, status, scatter
    per_part = 1 + 2 + 1 + 1 + levels + (w.m - 1) + 1 + 1 + 1 + 1
    launches_per_step = 3 + w.n_parts * per_part
    line = {
        "metric": METRIC_GRAPH, "value": ms, "unit": "ms", "n_gpus": rk.world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms, "higher_is_better": False, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic", "config": workload_config(args.workload),
        "status": int(res.status), "n_products": n_prod, "part_size": res.part_size, "core_size": res.core_size,
        "step_ms_min": float(min(step_ms)), "step_ms_max": float(max(step_ms)), "wall_s_timed_region": t_wall,
        "aggregate_solves_per_s": replicas_per_second(rk.world, ms),
        "e2e": {"value": e2e_ms, "unit": "ms", "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h),
                "steps": e2e_steps},
        "gpu_launches": launches_per_step * args.steps,
        "gpu_launches_note": f"{launches_per_step} per step: 3 halo kernels + {w.n_parts} parts x {per_part} (gather, "
                             f"2 Gershgorin, coefficients, map, {levels + w.m - 1} grouped product launches, partial sums, "
                             "trace, status, scatter)",
        "roofline": roof, "cpu_baseline": cpu, "clocks": clocks,
    }
    print(json.dumps(line), flush=True)
    rk.finish()
    return 0


# ----------------------------------------------------------------------------------------------------------
# our arm, graph-based workloads with SP2 as the local solver: one bml_graph_sp2_ellpack call per step
# ----------------------------------------------------------------------------------------------------------
def run_graph_sp2(args, rk=None, emit=True):
    """emit=False: return the JSON record instead of printing it (per_config of the default run; `rk` is the caller's)."""
    import torch

    from paper_2401_13772_b200 import api, hamiltonians as hm

    rk = rk or Ranks()
    api.load()
    dev = rk.dev
    w = hm.WORKLOADS[args.workload]
    H_np = hm.make_ellpack(args.workload)
    H_host = tuple(torch.from_numpy(a).pin_memory() for a in H_np)
    H_dev = tuple(a.to(dev) for a in H_host)
    offs_np, nodes_np = hm.regular_core_partition(w.N, w.n_parts)
    offs, nodes = torch.from_numpy(offs_np).to(dev), torch.from_numpy(nodes_np).to(dev)
    sizes = api.bml_graph_core_halo(H_dev, offs, nodes, w.graph_tol)[2].cpu().numpy()
    cap = int(sizes[:, 0].max())
    solver = api.GraphSp2Solver(w.N, w.M_out, w.n_parts, cap, dev)
    D_host = tuple(torch.empty_like(a).pin_memory() for a in (solver.dv.cpu(), solver.di.cpu(), solver.dn.cpu()))

    def solve(Hd):
        return solver.solve(Hd, offs, nodes, w.graph_tol, w.n_occ, w.idem_tol, w.drop_tol)

    step_ms, t_wall, clocks, res = timed_steps(rk, lambda: solve(H_dev), args)
    ms = float(np.mean(step_ms))

    def e2e_step():
        D, _ = solve(tuple(a.to(dev, non_blocking=True) for a in H_host))
        for dst, src in zip(D_host, D):
            dst.copy_(src, non_blocking=True)
        torch.cuda.synchronize()

    e2e_steps = max(3, min(args.steps, 10))
    h2d = sum(a.numel() * a.element_size() for a in H_host)
    d2h = sum(a.numel() * a.element_size() for a in D_host)
    e2e_ms = timed_e2e(rk, e2e_step, e2e_steps)

    # dominant kernel: x2_dense_fp64_batch_kernel, one launch = one product of every part; its rate is taken in-step
    # (the launches are the step but for the halo / gather / rescale / scatter kernels, < 1% of it)
    peak_probe = api.bml_probe_fp64_tensor_peak(40000)
    n_prod = int(res.sp2.n_products)
    flops = sum(dense_flops_per_product(int(sz)) if sz > 1024 else 2.0 * (((sz + 127) // 128) * ((sz + 127) // 128 + 1) // 2) * 128 * 128 * sz
                for sz in res.part_size)
    achieved = flops * n_prod / (ms * 1e-3) / 1e12
    roof = {
        "bound": "tensor", "kernel": "x2_dense_fp64_batch_kernel", "achieved": achieved, "peak": peak_probe,
        "unit": "TFLOP/s", "frac": achieved / peak_probe, "traffic": ncu_traffic(args.workload)["bytes"],
        "peak_source": "FP64 DMMA issue peak measured live by bml_probe_fp64_tensor_peak in this run "
                       "(MEASURED_PEAKS.json has no FP64 entry)",
        "note": "in-step rate: executed flops of all products / whole time-to-D (includes halo, gather, rescale, scatter)",
        "launch_ms": ms / max(n_prod, 1), "flops_per_launch": flops, "part_size": res.part_size,
    }
    ms, e2e_ms = aggregate_over_ranks([ms, e2e_ms], rk.dist, dev)
    if rk.rank != 0:
        rk.finish()
        return 0
    cpu = None
    if rk.world == 1 and not args.no_cpu_baseline:
        v, sample, cores = oracle_graph_sp2_time_to_D(args.workload, H_np, n_prod)
        cpu = {"value": v, "unit": "ms", "cores": cores, "kind": "oracle", "sample": sample}
    n_enq = 16
    while n_enq < 100:
        n_enq += 8
        if n_enq - 8 >= max(n_prod, 16):
            break
    # 3 halo kernels + 2 Gershgorin + per part (gather, rescale) + core trace + init + products + final buffers + scatters
    launches_per_step = 3 + 2 + 2 * w.n_parts + 2 + min(n_enq, 100) + 1 + w.n_parts
    line = {
        "metric": METRIC_GRAPH, "value": ms, "unit": "ms", "n_gpus": rk.world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms, "higher_is_better": False, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic", "config": workload_config(args.workload),
        "status": int(res.status), "n_products": n_prod, "branch": res.sp2.branch, "part_size": res.part_size,
        "core_size": res.core_size, "step_ms_min": float(min(step_ms)), "step_ms_max": float(max(step_ms)),
        "wall_s_timed_region": t_wall, "ms_per_product": ms / max(n_prod, 1),
        "aggregate_solves_per_s": replicas_per_second(rk.world, ms),
        "e2e": {"value": e2e_ms, "unit": "ms", "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h),
                "steps": e2e_steps},
        "gpu_launches": launches_per_step * args.steps,
        "gpu_launches_note": f"{launches_per_step} per step (upper bound): halo, Gershgorin, gather + rescale per part, "
                             f"{min(n_enq, 100)} batched product launches of which {n_prod} do work, scatter per part",
        "roofline": roof, "cpu_baseline": cpu, "clocks": clocks,
    }
    if not emit:
        return line
    print(json.dumps(line), flush=True)
    rk.finish()
    return 0


# ----------------------------------------------------------------------------------------------------------
# our arm, ELLBLOCK workloads: one bml_sp2_ellblock call per step
# ----------------------------------------------------------------------------------------------------------
def ellblock_block_macs(index, nnz, bs: int) -> int:
    """Executed multiply-adds of one upper-triangle block product: for every stored block (I, K), the blocks (K, J) with
    J >= I, bs^3 each (what kernel 1's DMMA chains execute for bs >= 8).  torch, chunked over block rows."""
    import torch

    NB, MB = index.shape
    live = torch.arange(MB, device=index.device).unsqueeze(0) < nnz.unsqueeze(1)
    total = 0
    for I0 in range(0, NB, 256):
        I1 = min(NB, I0 + 256)
        K = index[I0:I1].long()                                   # [r, MB]
        rows = index[K]                                           # [r, MB, MB] block columns of row K
        ok = live[K] & (rows >= torch.arange(I0, I1, device=index.device).view(-1, 1, 1))
        total += int((ok.sum(dim=2) * live[I0:I1]).sum().item())
    return total * bs ** 3


def run_ellblock(args, rk=None, emit=True):
    """emit=False: return the JSON record instead of printing it (per_config of the default run; `rk` is the caller's)."""
    import torch

    from paper_2401_13772_b200 import api, hamiltonians as hm

    rk = rk or Ranks()
    api.load()
    dev = rk.dev
    w = hm.WORKLOADS[args.workload]
    H_np = hm.make_ellblock(args.workload)
    H_host = tuple(torch.from_numpy(a).pin_memory() for a in H_np)
    H_dev = tuple(a.to(dev) for a in H_host)
    NB = w.N // w.bs
    solver = api.EllblockSolver(NB, w.MB, w.bs, dev)
    D_host = tuple(torch.empty_like(a).pin_memory() for a in H_host)

    def solve(Hd, mp=100):
        return solver.solve(*Hd, w.n_occ, w.idem_tol, w.drop_tol, mp)

    step_ms, t_wall, clocks, res = timed_steps(rk, lambda: solve(H_dev), args)
    ms = float(np.mean(step_ms))

    def e2e_step():
        D, _ = solve(tuple(a.to(dev, non_blocking=True) for a in H_host))
        for dst, src in zip(D_host, D):
            dst.copy_(src, non_blocking=True)
        torch.cuda.synchronize()

    e2e_steps = max(3, min(args.steps, 10))
    h2d = sum(a.numel() * a.element_size() for a in H_host)
    e2e_ms = timed_e2e(rk, e2e_step, e2e_steps) if res.status >= 0 else float("nan")

    # dominant kernels: one fused product on a mid-sequence iterate (X_5), timed alone
    roof, n_prod = None, int(res.n_products)
    if res.status >= 0:
        Xmid, _ = solve(H_dev, 6)
        Xmid = tuple(t.clone() for t in Xmid)
        out = tuple(torch.zeros_like(t) for t in Xmid)
        ws = api._workspace(api.load().bml_x2_ellblock_workspace_bytes(NB, w.MB, w.bs), dev)
        k_ms = time_alone(lambda: api.bml_x2_ellblock(Xmid, 1, w.drop_tol, out, ws), 5, warm=2)
        macs = ellblock_block_macs(Xmid[1], Xmid[2], w.bs)
        peak_probe = api.bml_probe_fp64_tensor_peak(40000)
        achieved = 2.0 * macs / (k_ms * 1e-3) / 1e12
        blocks = int(Xmid[2].sum().item())
        pk, pk_src = peaks()
        gathered = 2.0 * (macs / w.bs ** 3) * w.bs * w.bs * 8        # two operand blocks per block product
        roof = {
            "bound": "tensor", "kernel": "x2_ellblock_upper_kernel + x2_ellblock_assemble_kernel", "achieved": achieved,
            "peak": peak_probe, "unit": "TFLOP/s", "frac": achieved / peak_probe, "traffic": ncu_traffic(args.workload)["bytes"],
            "peak_source": "FP64 DMMA issue peak measured live by bml_probe_fp64_tensor_peak in this run",
            "note": "flops of ALL upper-triangle block products (2 bs^3 per block pair with a common block column) / time "
                    "of the two kernels; kernel 1's norm pre-screen does not execute the pairs of candidates that are "
                    "certain to be dropped (about a third on the 5' model), so the executed DMMA rate is lower; the operand "
                    "blocks come from L2 (2 flop per byte at bs = 8), so L2 latency and instruction issue, not the tensor "
                    "pipe, bound this kernel",
            "launch_ms": k_ms, "flops_per_launch": 2.0 * macs, "mean_blocks_per_block_row": blocks / NB,
            "stored_fill": None, "gathered_bytes": gathered, "gathered_gbs": gathered / (k_ms * 1e-3) / 1e9,
            "compulsory_bytes": 2.0 * blocks * (w.bs * w.bs * 8 + 4),
            "compulsory_frac_of_hbm": 2.0 * blocks * (w.bs * w.bs * 8 + 4) / (k_ms * 1e-3) / 1e9 / pk["hbm_gbs"],
        }
    ms, e2e_ms = aggregate_over_ranks([ms, e2e_ms], rk.dist, dev)
    if rk.rank != 0:
        rk.finish()
        return 0
    cpu = None
    if rk.world == 1 and not args.no_cpu_baseline:
        import oracle

        lo, hi = oracle.gershgorin_ellblock(*H_np)
        X0 = oracle.rescale_ellblock(*H_np, lo, hi)[:3]
        t0 = time.perf_counter()
        oracle.x2_ellblock(*X0, w.drop_tol)
        per = time.perf_counter() - t0
        cpu = {"value": per * max(n_prod, 1) * 1e3, "unit": "ms", "cores": oracle.omp_threads(), "kind": "oracle",
               "sample": f"one oracle block product (the first, on X_0: the sparsest of the solve) timed, x {n_prod} products"}
    n_enq = 16
    while n_enq < 100:
        n_enq += 8
        if n_enq - 8 >= max(n_prod, 16):
            break
    launches_per_step = 2 + 1 + 1 + 1 + 2 * min(n_enq, 100) + 1
    line = {
        "metric": METRIC, "value": ms, "unit": "ms", "n_gpus": rk.world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms, "higher_is_better": False, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic", "config": workload_config(args.workload),
        "status": int(res.status), "n_products": n_prod, "branch": res.branch,
        "max_blocks_per_block_row": [int(x) for x in res.max_row_nnz],
        "step_ms_min": float(min(step_ms)), "step_ms_max": float(max(step_ms)), "wall_s_timed_region": t_wall,
        "ms_per_product": ms / max(n_prod, 1), "aggregate_solves_per_s": replicas_per_second(rk.world, ms),
        "e2e": {"value": e2e_ms, "unit": "ms", "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(h2d),
                "steps": e2e_steps},
        "gpu_launches": launches_per_step * args.steps,
        "gpu_launches_note": f"{launches_per_step} per step (upper bound); a product is two kernels",
        "roofline": roof, "cpu_baseline": cpu, "clocks": clocks,
    }
    if not emit:
        return line
    print(json.dumps(line), flush=True)
    rk.finish()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=30)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default=DEFAULT_WORKLOAD)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--per-config", dest="per_config", action="store_true", default=None,
                    help="attach the other BASELINE.json configs as `per_config` (default: on for the default workload)")
    ap.add_argument("--no-per-config", dest="per_config", action="store_false")
    ap.add_argument("--per-config-list", default="", help="restrict per_config to these workloads (comma-separated)")
    ap.add_argument("--traffic-from", default=None, metavar="CSV",
                    help="no benchmark: parse an `ncu --page raw --csv` export and store the per-launch DRAM bytes of "
                         "--traffic-kernels under --workload in profiles/r02_traffic.json")
    ap.add_argument("--traffic-kernels", default="", help="comma-separated kernel-name substrings")
    ap.add_argument("--traffic-note", default="")
    ap.add_argument("--lanczos-steps", type=int, default=0,
                    help="SP2 workloads: tighten the Gershgorin bounds with K Lanczos steps (8..64); 0 = Gershgorin only, "
                         "the configuration BASELINE.json names")
    args = ap.parse_args()
    if args.traffic_from:
        write_traffic(args.traffic_from, args.workload, [k for k in args.traffic_kernels.split(",") if k], args.traffic_note)
        return 0
    if args.per_config is None:
        args.per_config = args.workload == DEFAULT_WORKLOAD and args.impl == "ours"
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.impl == "reference":
        return run_reference(args)
    from paper_2401_13772_b200 import hamiltonians as hm

    if hm.WORKLOADS[args.workload].kind == "cheby":
        return run_cheby(args)
    if hm.WORKLOADS[args.workload].kind == "graph":
        return run_graph(args)
    if hm.WORKLOADS[args.workload].kind == "graph_sp2":
        return run_graph_sp2(args)
    if hm.WORKLOADS[args.workload].kind == "ellblock":
        return run_ellblock(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
