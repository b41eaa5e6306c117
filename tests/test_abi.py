"""No-GPU checks of the boundary: libbmlsp2.so builds for sm_100a, loads, and exports every symbol that
include/bml_sp2.h declares; struct layouts of the binding match the header; the product package never imports the
oracle (and the oracle never imports the product)."""
import ctypes
import os
import re
import subprocess

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    names = set()
    inc = os.path.join(ROOT, "include")
    for f in sorted(os.listdir(inc)):
        if f.endswith(".h"):
            names |= set(re.findall(r"BML_API\s+[\w\s\*]+?\b(bml_\w+)\s*\(", open(os.path.join(inc, f)).read()))
    return sorted(names)


def test_header_declares_the_north_star_entry_points():
    names = _declared()
    for required in ("bml_sp2_dense", "bml_sp2_ellpack", "bml_gershgorin", "bml_trace", "bml_chebyshev_dense",
                     "bml_symm_ab_dense", "bml_graph_chebyshev_ellpack", "bml_graph_sp2_ellpack", "bml_sp2_ellblock"):
        assert required in names


def test_library_builds_loads_and_exports_every_declared_symbol():
    from paper_2401_13772_b200 import build

    path = build.build()
    lib = ctypes.CDLL(path)
    for name in _declared():
        assert hasattr(lib, name), f"{name} declared in include/*.h but not exported"
    lib.bml_version.restype = ctypes.c_char_p
    assert b"sm_100a" in lib.bml_version()
    lib.bml_status_string.restype = ctypes.c_char_p
    assert b"overflow" in lib.bml_status_string(-3)


def test_binding_lists_the_same_exports_and_struct_sizes():
    from paper_2401_13772_b200 import api

    assert sorted(api.EXPORTS) == _declared()
    # the ctypes mirrors must have the C layout of the header (checked against gcc's sizeof)
    src = r"""
    #include <stdio.h>
    #include "bml_graph.h"
    #include "bml_ellblock.h"
    int main(void){ printf("%zu %zu %zu %zu %zu %zu %zu %zu %zu %zu\n", sizeof(bml_matrix_t), sizeof(bml_sp2_params_t), sizeof(bml_sp2_stats_t),
                           sizeof(bml_cheb_params_t), sizeof(bml_cheb_stats_t), sizeof(bml_graph_params_t),
                           sizeof(bml_graph_stats_t), sizeof(bml_graph_sp2_params_t), sizeof(bml_graph_sp2_stats_t),
                           sizeof(bml_ellblock_t)); return 0; }
    """
    import tempfile

    exe = os.path.join(tempfile.mkdtemp(), "sizeof_probe")
    subprocess.run(["gcc", "-x", "c", "-", "-I", os.path.join(ROOT, "include"), "-o", exe], input=src.encode(), check=True)
    out = subprocess.run([exe], capture_output=True, check=True).stdout.split()
    os.remove(exe)
    assert [int(x) for x in out] == [ctypes.sizeof(api.bml_matrix_t), ctypes.sizeof(api.bml_sp2_params_t),
                                    ctypes.sizeof(api.bml_sp2_stats_t), ctypes.sizeof(api.bml_cheb_params_t),
                                    ctypes.sizeof(api.bml_cheb_stats_t), ctypes.sizeof(api.bml_graph_params_t),
                                    ctypes.sizeof(api.bml_graph_stats_t), ctypes.sizeof(api.bml_graph_sp2_params_t),
                                    ctypes.sizeof(api.bml_graph_sp2_stats_t), ctypes.sizeof(api.bml_ellblock_t)]


def test_sass_contains_the_blackwell_instructions():
    """The FP64 path must be DMMA tensor instructions fed by TMA, not scalar DFMA loops."""
    from paper_2401_13772_b200 import build

    sass = subprocess.run(["cuobjdump", "-sass", build.build()], capture_output=True, text=True).stdout
    assert "DMMA.8x8x4" in sass
    assert "UTMALDG" in sass
    # the mixed-precision path must be tcgen05 MMAs with TMEM accumulators read back by tcgen05.ld
    assert "UTCHMMA" in sass
    assert "LDTM" in sass
    # every kernel family of the three headers is in the image
    for kernel in ("x2_dense_fp64_sk_kernel", "x2_dense_mixed_kernel", "x2_ellpack_upper_kernel", "symm_ab_fp64_kernel",
                   "cheb_coeff_kernel", "cheb_sums_kernel", "graph_gather_kernel", "graph_scatter_kernel",
                   "lanczos_run_kernel", "x2_dense_fp64_batch_kernel", "x2_ellblock_upper_kernel",
                   "x2_ellblock_assemble_kernel"):
        assert kernel in sass, kernel


def test_product_and_oracle_do_not_import_each_other():
    pkg = os.path.join(ROOT, "paper_2401_13772_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", text, re.M), f
                assert "sp2_oracle" not in text and "liboracle" not in text, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            text = open(os.path.join(ROOT, "oracle", f)).read()
            assert not re.search(r"^\s*(import|from)\s+paper_2401_13772_b200\b", text, re.M), f
            assert "libbmlsp2" not in text.replace("libbmlsp2.so, ", "") or f == "__init__.py"


def test_api_refuses_cpu_tensors():
    import pytest
    import torch

    from paper_2401_13772_b200 import api

    with pytest.raises(RuntimeError):
        api.bml_sp2_dense(torch.eye(4, dtype=torch.float64), 2, 1e-10)
