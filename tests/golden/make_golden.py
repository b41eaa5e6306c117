#!/usr/bin/env python
"""Writes tests/golden/sp2_expected.json -- the stored expected values of the parity tests.

    python tests/golden/make_golden.py [workload ...]        (default: every workload listed in CASES)

Every stored value is produced by the CPU oracle (oracle/sp2_oracle.c) on the seeded synthetic Hamiltonians of
paper_2401_13772_b200/hamiltonians.py; nothing here imports, loads or runs the CUDA path.  The paper itself prints
no worked numeric example for SP2 (PAPER.md P:155-212 gives Eq. 5-7 and Listing 2 only; its "22 iterations",
P:171, needs the bio-benchmark Hamiltonians, which are not available), so there is no paper-printed fixture.

Stored per case: Gershgorin bounds, status, m*, number of products, the branch string b_0..b_{m*-1}
(Eq. 6-7), tr X_m and e_m per product, and a few entries / the trace / Frobenius norm of D.
The N=8192 case takes the oracle ~10-20 minutes on 8 cores (32 naive N^3 products); the others take seconds.
"""
from __future__ import annotations

import json
import os
import sys
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import oracle  # noqa: E402
from paper_2401_13772_b200 import hamiltonians as hm  # noqa: E402  (input generators only)

OUT = os.path.join(HERE, "sp2_expected.json")
CASES = ["dense_n256", "dense_n2048", "dense_n8192", "ellpack_small_12x10x8"]
SAMPLE = [(0, 0), (0, 1), (1, 0), (5, 17), (100, 100), (127, 128), (128, 127), (255, 255)]


def dense_case(name):
    w = hm.WORKLOADS[name]
    H = hm.make_dense(name)
    D, st = oracle.sp2_dense(H, w.n_occ, w.idem_tol)
    N = w.N
    samp = [(i % N, j % N) for i, j in SAMPLE] + [(N - 1, 0), (N // 2, N // 2 - 1)]
    return {
        "kind": "dense", "N": N, "n_occ": w.n_occ, "idem_tol": w.idem_tol,
        "emin": st["emin"], "emax": st["emax"], "status": st["status"], "m_star": st["m_star"],
        "n_products": st["n_products"], "branch": st["branch"],
        "trace": [float(x) for x in st["trace"]], "idem": [float(x) for x in st["idem"]],
        "D_trace": float(np.trace(D)), "D_fro": float(np.linalg.norm(D)),
        "D_samples": [[i, j, float(D[i, j])] for i, j in samp],
    }


def ellpack_small_case():
    L, M, tau, tol = (12, 10, 8), 512, 1e-6, 1e-8
    Hs = hm.small_sparse_model(L, M=M)
    n = Hs[0].shape[0]
    (dv, di, dn), st = oracle.sp2_ellpack(*Hs, n // 2, tol, tau)
    return {
        "kind": "ellpack", "lattice": list(L), "N": n, "M": M, "n_occ": n // 2, "idem_tol": tol, "drop_tol": tau,
        "emin": st["emin"], "emax": st["emax"], "status": st["status"], "m_star": st["m_star"],
        "n_products": st["n_products"], "branch": st["branch"],
        "trace": [float(x) for x in st["trace"]], "idem": [float(x) for x in st["idem"]],
        "max_row_nnz": [int(x) for x in st["max_row_nnz"]],
        "D_nnz_total": int(dn.sum()), "D_row0_index": [int(x) for x in di[0, : dn[0]]],
        "D_row0_value": [float(x) for x in dv[0, : dn[0]]],
    }


def main():
    todo = sys.argv[1:] or CASES
    data = json.load(open(OUT)) if os.path.exists(OUT) else {}
    for name in todo:
        t0 = time.time()
        data[name] = ellpack_small_case() if name == "ellpack_small_12x10x8" else dense_case(name)
        data[name]["oracle_seconds"] = round(time.time() - t0, 1)
        data[name]["oracle_threads"] = oracle.omp_threads()
        print(f"{name}: products={data[name]['n_products']} branch={data[name]['branch']} "
              f"({data[name]['oracle_seconds']} s)", flush=True)
        with open(OUT, "w") as f:
            json.dump(data, f, indent=1, sort_keys=True)
            f.write("\n")


if __name__ == "__main__":
    main()
