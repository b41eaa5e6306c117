"""CPU check of the inequality the sparse kernels' exact pre-screens rest on, against the oracle's
products -- no GPU, no kernel code: restated here in numpy.

ELLPACK (scalar): for a 32-column block B,  |P_ij| <= sum_k |x_ik| max_{j' in B} |x_kj'|  for every j in B, so a block whose
bound is below tau holds only entries that thr() drops.  ELLBLOCK: ||P_IJ||_F <= sum_K ||X_IK||_F ||X_JK||_F.
The kernels skip what falls below tau (1 - margin); the tests check on the oracle's own P = thr(X X) that no kept entry /
block lies in a skipped block / below the bound -- i.e. that skipping cannot change the oracle's result."""
import numpy as np
import pytest

from paper_2401_13772_b200 import hamiltonians as hm


def _x0(oracle_mod, H):
    lo, hi = oracle_mod.gershgorin_ellpack(*H)
    return oracle_mod.rescale_ellpack(*H, lo, hi)[:3]


@pytest.mark.parametrize("tau", [1e-6, 1e-4, 1e-2])
def test_no_kept_entry_of_the_oracles_product_lies_in_a_screened_column_block(oracle_mod, tau):
    H = hm.small_sparse_model((12, 10, 8), M=512)
    X = _x0(oracle_mod, H)
    # second iterate too: wider rows, mixed magnitudes
    P0 = oracle_mod.x2_ellpack(*X, tau)[:3]
    X1 = oracle_mod.update_ellpack(X, P0, tau)[:3]
    n_skipped_touched = 0
    for Xm in (X, X1):
        Xd = hm.ellpack_to_dense(*Xm)
        N = Xd.shape[0]
        pv, pi, pn = oracle_mod.x2_ellpack(*Xm, tau)[:3]
        nb = (N + 31) // 32
        pad = nb * 32 - N
        A = np.abs(np.pad(Xd, ((0, 0), (0, pad))))
        blockmax = A.reshape(N, nb, 32).max(axis=2)                   # [k, B] = max_{j in B} |x_kj|
        bound = np.abs(Xd) @ blockmax                                 # [i, B] = sum_k |x_ik| blockmax[k, B]
        skipped = bound < tau * (1.0 - 1e-3)                          # what the kernel does not accumulate
        for i in range(N):
            cols = pi[i, : pn[i]]
            offdiag = cols[cols != i]
            assert not skipped[i, offdiag // 32].any(), (i, tau)
            # and the bound really is one: every stored value, kept or not, is below it
            assert (np.abs(pv[i, : pn[i]]) <= bound[i, cols // 32] * (1 + 1e-12) + 1e-300).all()
            n_skipped_touched += int((skipped[i] & (bound[i] > 0)).sum())
    assert n_skipped_touched > 0, "the case must exercise the screen"


@pytest.mark.parametrize("bs", [4, 8])
def test_no_kept_block_of_the_oracles_block_product_is_below_the_norm_bound(oracle_mod, bs):
    tau = 1e-6
    Hs = hm.small_sparse_model((8, 8, 16), M=512)
    N = Hs[0].shape[0]
    H = hm.ellblock_from_ellpack(*Hs, bs, N // bs)
    lo, hi = oracle_mod.gershgorin_ellblock(*H)
    X = oracle_mod.rescale_ellblock(*H, lo, hi)[:3]
    pv, pi, pn = oracle_mod.x2_ellblock(*X, tau)[:3]
    NB = N // bs
    Xd = hm.ellblock_to_dense(*X)
    nrm = np.sqrt((Xd.reshape(NB, bs, NB, bs) ** 2).sum(axis=(1, 3)))   # [I, K] = ||X_IK||_F (0 where absent)
    bound = nrm @ nrm.T                                                  # sum_K ||X_IK|| ||X_JK||
    pv = pv.reshape(NB, -1, bs, bs)
    skipped = 0
    for I in range(NB):
        for q in range(pn[I]):
            J = pi[I, q]
            assert np.linalg.norm(pv[I, q]) <= bound[I, J] * (1 + 1e-12)
            if J != I:
                assert bound[I, J] >= tau * (1.0 - 1e-9)
        skipped += int(((bound[I] > 0) & (bound[I] < tau * (1.0 - 1e-4))).sum())
    assert skipped > 0, "the case must exercise the screen"
