"""The boundary as a C programmer sees it: a plain C caller built with gcc against include/bml_sp2.h and
linked to libbmlsp2.so, argument checks that never reach CUDA, the asynchronous stats == NULL form, the cached-state
release, and the split between the product headers and include/bml_sp2_testing.h."""
import ctypes
import os
import re
import subprocess
import tempfile

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
INC = os.path.join(ROOT, "include")
CUDA = os.environ.get("CUDA_HOME", "/usr/local/cuda")


@pytest.fixture(scope="module")
def c_caller():
    from paper_2401_13772_b200 import build

    lib = build.build()
    exe = os.path.join(tempfile.mkdtemp(), "abi_smoke")
    cmd = ["gcc", "-std=c99", "-Wall", "-Werror", "-O1", os.path.join(ROOT, "tests", "c", "abi_smoke.c"), "-I", INC,
           "-I", os.path.join(CUDA, "include"), "-o", exe, lib, "-L", os.path.join(CUDA, "lib64"), "-lcudart", "-lm",
           "-Wl,-rpath," + os.path.dirname(lib), "-Wl,-rpath," + os.path.join(CUDA, "lib64")]
    subprocess.run(cmd, check=True)
    return exe


def test_c_caller_builds_against_the_product_header_and_checks_arguments(c_caller):
    out = subprocess.run([c_caller, "--no-gpu"], capture_output=True, text=True)
    assert out.returncode == 0 and "OK no-gpu" in out.stdout, out.stdout + out.stderr


@pytest.mark.gpu
def test_c_caller_solves_on_the_gpu_without_python(c_caller):
    out = subprocess.run([c_caller], capture_output=True, text=True)
    assert out.returncode == 0 and "OK gpu" in out.stdout, out.stdout + out.stderr


def test_product_headers_hold_no_test_hooks():
    hooks = ("bml_probe_fp64_tensor_peak", "bml_dense_work_item", "bml_dense_mixed_tile_count",
             "bml_dense_mixed_tile_of_cta", "bml_symm_work_item", "bml_cheb_schedule")
    testing = open(os.path.join(INC, "bml_sp2_testing.h")).read()
    for name in hooks:
        assert re.search(r"BML_API[^;]*\b%s\s*\(" % name, testing), name
        for h in ("bml_sp2.h", "bml_chebyshev.h", "bml_graph.h"):
            assert name not in open(os.path.join(INC, h)).read(), (name, h)


def test_mixed_single_product_rejects_a_pitch_the_workspace_was_not_sized_for():
    """bml_x2_dense_workspace_bytes(N, precision) sizes the 16-bit planes for ld = 16 ceil(N / 16); a wider
    ld used to pass the argument check and overrun the workspace.  The check sits before any CUDA call."""
    from paper_2401_13772_b200 import api

    L = api.load()
    N, ld = 1000, 1024                       # 16 * ceil(1000 / 16) = 1008: ld = 1024 is a multiple of 16 but too wide
    nbytes = L.bml_x2_dense_workspace_bytes(N, 1)
    x = api.bml_matrix_t(api.BML_DENSE, 0, N, ld, 0x10000, None, None)
    xn = api.bml_matrix_t(api.BML_DENSE, 0, N, ld, 0x4000000, None, None)
    for precision in (1, 2):
        rc = L.bml_x2_dense(ctypes.byref(x), ctypes.byref(xn), 1, precision, ctypes.c_void_p(0x800),
                            ctypes.c_void_p(0x400), L.bml_x2_dense_workspace_bytes(N, precision), None)
        assert rc == -1
    assert nbytes > 2 * 2 * N * 1008 * 2     # two plane sets of two 16-bit planes at the pitch the check enforces


@pytest.mark.gpu
def test_asynchronous_solve_reads_its_verdict_later():
    import torch

    from paper_2401_13772_b200 import api, hamiltonians as hm

    H = torch.from_numpy(hm.make_dense("dense_n256")).cuda()
    solver = api.DenseSolver(256, H.device)
    D1, r1 = solver.solve(H, 128, 1e-10)
    D1 = D1.clone()
    D2, none = solver.solve(H, 128, 1e-10, asynchronous=True)
    assert none is None
    r2 = solver.read_stats()
    assert (r2.status, r2.n_products, r2.branch) == (r1.status, r1.n_products, r1.branch)
    assert torch.equal(D1, D2)
    api.bml_sp2_release_cached()
    D3, r3 = solver.solve(H, 128, 1e-10)
    assert torch.equal(D1, D3) and r3.branch == r1.branch


@pytest.mark.gpu
def test_failed_solve_leaves_D_untouched():
    import torch

    from paper_2401_13772_b200 import api

    H = (3.0 * torch.eye(64, dtype=torch.float64)).cuda()          # H = c I: degenerate bounds, status -2
    solver = api.DenseSolver(64, H.device)
    solver.D.fill_(7.0)
    D, res = solver.solve(H, 32, 1e-10)
    assert res.status == -2
    assert bool((D == 7.0).all())
