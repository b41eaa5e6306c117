"""Host-side checks of the work distribution of the dense kernels (no GPU): the library exports the very arithmetic its
kernels run (bml_dense_work_item, bml_dense_mixed_tile_of_cta), and these tests check that every (tile, k-slab) unit of
the upper triangle is covered exactly once, that split tiles have exactly one owner (the part that starts at k-slab 0)
and that contributors are the CTAs right after it -- the assumptions the stream-K hand-off rests on."""
import pytest

from paper_2401_13772_b200 import api


@pytest.mark.parametrize("N,G", [(1100, 148), (2048, 148), (2048, 132), (3000, 148), (8192, 148), (1283, 7), (4096, 1)])
def test_persistent_fp64_work_list_covers_every_unit_once(N, G):
    T = (N + 127) // 128
    KT = (N + 15) // 16
    tiles = T * (T + 1) // 2
    cover = {}
    per_cta = []
    for c in range(G):
        items = api.bml_dense_work_items(N, G, c)
        per_cta.append(items)
        n_contrib = 0
        for tile, I, J, k0, k1 in items:
            assert 0 <= I <= J < T and tile == J * (J + 1) // 2 + I
            assert 0 <= k0 < k1 <= KT
            cover.setdefault(tile, []).append((k0, k1, c))
            n_contrib += k0 > 0
        assert n_contrib <= 1, "a CTA has one scratch slot: at most one contributed partial per launch"
    assert sorted(cover) == list(range(tiles))
    for tile, parts in cover.items():
        parts.sort()
        assert parts[0][0] == 0 and parts[-1][1] == KT
        for (a0, a1, ca), (b0, b1, cb) in zip(parts, parts[1:]):
            assert a1 == b0, "k ranges of a split tile must tile [0, KT) without gap or overlap"
            assert cb > ca, "contributors are later CTAs than the owner, in ascending order"
        owner = parts[0][2]
        assert [p[2] for p in parts] == list(range(owner, owner + len(parts)))
    # balance: every CTA runs the same number of full tiles, and the split wave differs by at most one k-slab
    units = [sum(k1 - k0 for _, _, _, k0, k1 in items) for items in per_cta]
    W = tiles // G
    tail = [u - W * KT for u in units]
    assert max(tail) - min(tail) <= 1


@pytest.mark.parametrize("N", [1, 128, 129, 3072, 3073, 5000, 16384])
def test_mixed_tile_map_is_a_bijection_onto_the_upper_triangle(N):
    T = (N + 127) // 128
    tiles = [t for t in api.bml_dense_mixed_tiles(N) if t is not None]
    assert len(tiles) == len(set(tiles)) == T * (T + 1) // 2
    assert all(0 <= I <= J < T for I, J in tiles)


def test_work_item_rejects_bad_arguments():
    import ctypes

    L = api.load()
    out = (ctypes.c_int32 * 5)()
    assert L.bml_dense_work_item(512, 148, 0, 0, out) == -1       # small matrices do not use the persistent kernel
    assert L.bml_dense_work_item(2048, 148, 148, 0, out) == -1
    assert L.bml_dense_work_item(2048, 148, 0, 0, None) == -1
