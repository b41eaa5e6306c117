"""GPU test of include/bml_no_alloc.h: bml_gershgorin_static (scratch in a static device array of the library; for
callers that cannot allocate) against the existing bml_gershgorin path (caller-supplied workspace).  Both launch the same
kernels with the same summation order, so the bounds must be bit-identical -- the bar tests/test_gpu_dense.py and
tests/test_gpu_ellpack.py hold bml_gershgorin itself to against the oracle.

Collected last on purpose (file name): the suite runs with `pytest -x`, and a failure here must not hide another test.
Runs alone in a fresh process (the first call resolves the array's device address) and after the other tests."""
import numpy as np
import pytest

from paper_2401_13772_b200 import hamiltonians as hm

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def api():
    import torch

    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2401_13772_b200 import api as a

    a.load()
    return a


def _dense(name):
    import torch

    return torch.from_numpy(np.ascontiguousarray(hm.make_dense(name))).cuda()


def test_static_gershgorin_matches_the_workspace_path_on_two_calls_in_a_row(api):
    import torch

    big = _dense("dense_n2048")
    small = _dense("dense_n256")
    out = torch.full((2,), float("nan"), dtype=torch.float64, device="cuda")
    # two calls in a row on the same matrix, then a smaller one (the scratch still holds the rows of the larger one
    # beyond its N: they must not be read), then the larger one again
    for H in (big, big, small, big):
        ref = api.bml_gershgorin(H)
        out.fill_(float("nan"))
        got = api.bml_gershgorin_static(H, out)
        torch.cuda.synchronize()
        assert torch.equal(got, ref), (got.tolist(), ref.tolist())
        assert got[0].item() < got[1].item()


def test_static_gershgorin_ellpack_and_strided_dense(api):
    import torch

    value, index, nnz = hm.make_ellpack("ellpack_n65536")        # N = 65536 = BML_GERSHGORIN_STATIC_MAX_N exactly
    ell = (torch.from_numpy(value).cuda(), torch.from_numpy(index).cuda(), torch.from_numpy(nnz).cuda())
    assert ell[0].shape[0] == api.GERSHGORIN_STATIC_MAX_N
    out = torch.empty(2, dtype=torch.float64, device="cuda")
    for _ in range(2):
        ref = api.bml_gershgorin(ell)
        got = api.bml_gershgorin_static(ell, out)
        torch.cuda.synchronize()
        assert torch.equal(got, ref)
    # a dense matrix with a row pitch larger than N
    Hp = api.padded_dense(hm.make_dense("dense_n256"))
    assert torch.equal(api.bml_gershgorin_static(Hp, out), api.bml_gershgorin(Hp))


def test_static_gershgorin_allocates_nothing_and_rejects_large_n(api):
    import ctypes

    import torch

    H = _dense("dense_n256")
    out = torch.empty(2, dtype=torch.float64, device="cuda")
    api.bml_gershgorin_static(H, out)                  # first call on the device: address lookup, lazy module load
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    torch_bytes0 = torch.cuda.memory_reserved()
    for _ in range(3):
        api.bml_gershgorin_static(H, out)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0 and torch.cuda.memory_reserved() == torch_bytes0
    # one row more than the static scratch holds: refused with its own status, nothing launched, `out` untouched
    N = api.GERSHGORIN_STATIC_MAX_N + 1
    value = torch.ones((N, 1), dtype=torch.float64, device="cuda")
    index = torch.arange(N, dtype=torch.int32, device="cuda").reshape(N, 1).contiguous()
    nnz = torch.ones(N, dtype=torch.int32, device="cuda")
    before = out.clone()
    L = api.load()
    desc = api.ellpack_desc(value, index, nnz)
    rc = L.bml_gershgorin_static(ctypes.byref(desc), out.data_ptr(), None)
    assert rc == -8
    assert b"BML_GERSHGORIN_STATIC_MAX_N" in L.bml_no_alloc_status_string(rc)
    assert L.bml_no_alloc_status_string(-3) == L.bml_status_string(-3)
    with pytest.raises(RuntimeError, match="static scratch"):
        api.bml_gershgorin_static((value, index, nnz), out)
    torch.cuda.synchronize()
    assert torch.equal(out, before)
    # the workspace path serves the same matrix
    assert api.bml_gershgorin((value, index, nnz)).tolist() == [1.0, 1.0]
