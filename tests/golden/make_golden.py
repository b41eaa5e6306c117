#!/usr/bin/env python
"""Writes tests/golden/sp2_expected.json -- the stored expected values of the parity tests.

    python tests/golden/make_golden.py [workload ...]        (default: every workload listed in CASES)

Every stored value is produced by the CPU oracle (oracle/sp2_oracle.c) on the seeded synthetic Hamiltonians of
paper_2401_13772_b200/hamiltonians.py; nothing here imports, loads or runs the CUDA path.  The paper itself prints
no worked numeric example for SP2 (PAPER.md P:155-212 gives Eq. 5-7 and Listing 2 only; its "22 iterations",
P:171, needs the bio-benchmark Hamiltonians, which are not available), so there is no paper-printed fixture.

Stored per case: Gershgorin bounds, status, m*, number of products, the branch string b_0..b_{m*-1}
(Eq. 6-7), tr X_m and e_m per product, and a few entries / the trace / Frobenius norm of D.
The full-size dense cases also store the whole-matrix probe y = D v for the seeded Gaussian vector v = probe_vector(N)
(E ||A v||^2 = ||A||_F^2, so ||D_gpu v - y|| estimates ||D_gpu - D_oracle||_F over EVERY entry of D); the arrays go to
tests/golden/<case>_Dv.txt (one value per line, repr precision).  The full-size ELLPACK case stores a SHA-256 over the
(value, index, nnz) arrays of D restricted to the stored entries, plus 16 whole rows.

Cost on 8 cores: dense_n8192 (32 naive N^3 products) and mixed_n16384_first4 (the FP64 oracle stopped after 4 products
at N=16384: the reference for the mixed-precision kernel's X_3) ~15-30 min each; ellpack_n65536 (the 12-product 5'
solve) ~1-2 min; the others seconds.  `mixed_n16384` (not in the default list: the full 30-product FP64 oracle solve of
configs[3], 1.3e14 multiply-adds) takes hours.
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
CASES = ["dense_n256", "dense_n2048", "dense_n8192", "ellpack_small_12x10x8", "ellpack_n65536", "mixed_n16384_first4",
         "ellblock_n65536"]
PROBE_SEED = 20240126          # the paper's date; any fixed seed does
SAMPLED_ROWS = 16
SAMPLE = [(0, 0), (0, 1), (1, 0), (5, 17), (100, 100), (127, 128), (128, 127), (255, 255)]


def probe_vector(N):
    """Seeded Gaussian probe vector (an input: the tests rebuild it with the same two lines)."""
    return np.random.default_rng(PROBE_SEED).standard_normal(N)


def write_vector(name, y):
    with open(os.path.join(HERE, name), "w") as f:
        f.write("".join(repr(float(v)) + "\n" for v in y))


def dense_case(name, max_products=100, workload=None):
    w = hm.WORKLOADS[workload or name]
    H = hm.make_dense(workload or name)
    D, st = oracle.sp2_dense(H, w.n_occ, w.idem_tol, max_products=max_products)
    N = w.N
    samp = [(i % N, j % N) for i, j in SAMPLE] + [(N - 1, 0), (N // 2, N // 2 - 1)]
    extra = {}
    if N >= 4096:
        rng = np.random.default_rng(PROBE_SEED + 1)
        samp += [(int(i), int(j)) for i, j in zip(rng.integers(0, N, 64), rng.integers(0, N, 64))]
        write_vector(name + "_Dv.txt", D @ probe_vector(N))
        extra = {"Dv_file": name + "_Dv.txt", "probe_seed": PROBE_SEED, "max_products": max_products,
                 "workload": workload or name}
    return {
        **extra,
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


def ell_digest(dv, di, dn):
    """SHA-256 over nnz[N] (int32) then, row by row, the stored columns (int32) and values (float64 bit patterns)."""
    import hashlib

    h = hashlib.sha256()
    h.update(np.ascontiguousarray(dn, dtype=np.int32).tobytes())
    keep = np.arange(dv.shape[1])[None, :] < dn[:, None]
    h.update(np.ascontiguousarray(di[keep], dtype=np.int32).tobytes())
    h.update(np.ascontiguousarray(dv[keep], dtype=np.float64).tobytes())
    return h.hexdigest()


def ellpack_full_case(name):
    w = hm.WORKLOADS[name]
    Hs = hm.make_ellpack(name)
    (dv, di, dn), st = oracle.sp2_ellpack(*Hs, w.n_occ, w.idem_tol, w.drop_tol)
    rows = [int(r) for r in np.random.default_rng(PROBE_SEED).integers(0, w.N, SAMPLED_ROWS - 2)] + [0, w.N - 1]
    return {
        "kind": "ellpack", "workload": name, "N": w.N, "M": w.M, "n_occ": w.n_occ, "idem_tol": w.idem_tol,
        "drop_tol": w.drop_tol,
        "emin": st["emin"], "emax": st["emax"], "status": st["status"], "m_star": st["m_star"],
        "n_products": st["n_products"], "branch": st["branch"],
        "trace": [float(x) for x in st["trace"]], "idem": [float(x) for x in st["idem"]],
        "max_row_nnz": [int(x) for x in st["max_row_nnz"]],
        "D_nnz_total": int(dn.sum()), "D_nnz_max": int(dn.max()), "D_sha256": ell_digest(dv, di, dn),
        "D_trace": float(oracle.trace_ellpack(dv, di, dn)),
        "D_rows": [{"row": r, "index": [int(x) for x in di[r, : dn[r]]],
                    "value": [float(x) for x in dv[r, : dn[r]]]} for r in rows],
    }


def ellblock_matvec(dv, di, dn, v):
    """y = D v for D in ELLBLOCK form (numpy; the GPU test does the same product with torch on its own D)."""
    NB, MB, bs, _ = dv.shape
    live = (np.arange(MB)[None, :] < dn[:, None])[:, :, None, None]
    y = np.zeros((NB, bs))
    vb = v.reshape(NB, bs)
    for I0 in range(0, NB, 512):
        I1 = min(NB, I0 + 512)
        y[I0:I1] = np.einsum("ipab,ipb->ia", dv[I0:I1] * live[I0:I1], vb[di[I0:I1]])
    return y.reshape(-1)


def ellblock_full_case(name):
    """SURVEY 8(f) f-4 at BASELINE size: the ELLBLOCK oracle's whole solve of the 5' model in bs x bs blocks."""
    w = hm.WORKLOADS[name]
    H = hm.make_ellblock(name)
    (dv, di, dn), st = oracle.sp2_ellblock(*H, w.n_occ, w.idem_tol, w.drop_tol, 100)
    NB = dv.shape[0]
    dv4 = dv.reshape(NB, w.MB, w.bs, w.bs)
    live = np.arange(w.MB)[None, :] < dn[:, None]
    write_vector(name + "_Dv.txt", ellblock_matvec(dv4, di, dn, probe_vector(w.N)))
    rows = [int(r) for r in np.random.default_rng(PROBE_SEED).integers(0, NB, 6)] + [0, NB - 1]
    return {
        "kind": "ellblock", "workload": name, "N": w.N, "bs": w.bs, "MB": w.MB, "n_occ": w.n_occ, "idem_tol": w.idem_tol,
        "drop_tol": w.drop_tol, "Dv_file": name + "_Dv.txt", "probe_seed": PROBE_SEED,
        "emin": st["emin"], "emax": st["emax"], "status": st["status"], "m_star": st["m_star"],
        "n_products": st["n_products"], "branch": st["branch"],
        "trace": [float(x) for x in st["trace"]], "idem": [float(x) for x in st["idem"]],
        "max_row_nnz": [int(x) for x in st["max_row_nnz"]],
        "D_blocks_total": int(dn.sum()), "D_blocks_max": int(dn.max()),
        "D_fro": float(np.sqrt((dv4[live] ** 2).sum())), "D_trace": float(oracle.trace_ellblock(dv, di, dn)),
        "D_rows": [{"row": r, "index": [int(x) for x in di[r, : dn[r]]],
                    "block_norm": [float(np.linalg.norm(dv4[r, q])) for q in range(dn[r])]} for r in rows],
    }


def run_case(name):
    if name.startswith("ellblock_"):
        return ellblock_full_case(name)
    if name == "ellpack_small_12x10x8":
        return ellpack_small_case()
    if name == "ellpack_n65536":
        return ellpack_full_case(name)
    if name == "mixed_n16384_first4":
        # the FP64 oracle on configs[3]'s input, stopped by S3 after 4 products: D = X_3 (reading 6), status 2
        return dense_case(name, max_products=4, workload="mixed_n16384")
    # "mixed_n16384": reading 17 -- the oracle of the mixed-precision mode is the FP64 oracle at the mixed config's
    # tolerance (1e-6); ~30 naive products at N = 16384, hours on 8 cores: run on request only
    return dense_case(name)


def main():
    todo = sys.argv[1:] or CASES
    data = json.load(open(OUT)) if os.path.exists(OUT) else {}
    for name in todo:
        t0 = time.time()
        case = run_case(name)
        data = json.load(open(OUT)) if os.path.exists(OUT) else {}      # re-read: cases may be run side by side
        data[name] = case
        data[name]["oracle_seconds"] = round(time.time() - t0, 1)
        data[name]["oracle_threads"] = oracle.omp_threads()
        print(f"{name}: products={data[name]['n_products']} branch={data[name]['branch']} "
              f"({data[name]['oracle_seconds']} s)", flush=True)
        with open(OUT, "w") as f:
            json.dump(data, f, indent=1, sort_keys=True)
            f.write("\n")


if __name__ == "__main__":
    main()
