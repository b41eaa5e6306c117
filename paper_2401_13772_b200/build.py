"""Build libbmlsp2.so (hand-written sm_100a CUDA + the C ABI of include/*.h) in-tree with nvcc.

    python -m paper_2401_13772_b200.build [--force] [--verbose]

nvcc cross-compiles without a GPU.  The library is written next to this file so that it travels with the repo
snapshot to the GPU box; it is git-ignored (history stays source-only).
"""
from __future__ import annotations

import os
import subprocess
import sys

_HERE = os.path.dirname(os.path.abspath(__file__))
_CSRC = os.path.join(_HERE, "csrc")
_INC = os.path.join(os.path.dirname(_HERE), "include")
LIB_PATH = os.path.join(_HERE, "libbmlsp2.so")
SOURCES = ["api.cu", "dense_fp64.cu", "dense_mixed.cu", "ellpack.cu", "reductions.cu", "gershgorin_static.cu", "probe.cu", "symm_ab.cu",
           "chebyshev.cu", "graph.cu", "bounds.cu", "dense_batch.cu", "ellblock.cu"]
NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17", "-Xcompiler", "-fPIC",
    "-Xcompiler", "-fvisibility=hidden", "--expt-relaxed-constexpr", "-fmad=true",
]
# extra nvcc flags for kernel experiments (e.g. BML_NVCC_EXTRA="-DBML_ELL_BUCKET_LOG2=3"); empty in normal builds
NVCC_FLAGS += os.environ.get("BML_NVCC_EXTRA", "").split()


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def _stale() -> bool:
    if not os.path.exists(LIB_PATH):
        return True
    t = os.path.getmtime(LIB_PATH)
    deps = [os.path.join(_CSRC, f) for f in os.listdir(_CSRC)] + [os.path.join(_INC, f) for f in os.listdir(_INC)] + [__file__]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    if not (force or _stale()):
        return LIB_PATH
    objs = []
    procs = []
    for src in SOURCES:
        obj = os.path.join(_CSRC, src.replace(".cu", ".o"))
        cmd = [_nvcc(), *NVCC_FLAGS, "-I", _INC, "-c", os.path.join(_CSRC, src), "-o", obj]
        if verbose:
            cmd.insert(1, "-Xptxas=-v")
            print(" ".join(cmd), flush=True)
        procs.append((src, subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)))
        objs.append(obj)
    failed = False
    for src, p in procs:
        out, _ = p.communicate()
        if p.returncode != 0 or verbose:
            print(f"--- {src}\n{out}", flush=True)
        failed |= p.returncode != 0
    if failed:
        raise RuntimeError("nvcc failed")
    link = [_nvcc(), "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", LIB_PATH, *objs,
            "-Xlinker", "--exclude-libs,ALL"]
    subprocess.run(link, check=True)
    return LIB_PATH


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
