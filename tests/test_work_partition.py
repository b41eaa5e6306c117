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
    where = {}
    for c in range(G):
        items = api.bml_dense_work_items(N, G, c)
        per_cta.append(items)
        n_contrib = 0
        for tile, I, J, k0, k1 in items:
            # tile number -> (I, J) is a bijection onto the upper triangle (super-block order above 24 tile rows)
            assert 0 <= I <= J < T and where.setdefault(tile, (I, J)) == (I, J)
            if T <= 24:
                assert tile == J * (J + 1) // 2 + I
            assert 0 <= k0 < k1 <= KT
            cover.setdefault(tile, []).append((k0, k1, c))
            n_contrib += k0 > 0
        assert n_contrib <= 1, "a CTA has one scratch slot: at most one contributed partial per launch"
    assert sorted(cover) == list(range(tiles))
    assert len(set(where.values())) == tiles
    if T > 24:      # a wave of consecutive tiles shares few row panels: at most 2 x 12 + a super-block boundary
        wave = [where[t] for t in range(min(G, tiles))]
        assert len({i for i, _ in wave} | {j for _, j in wave}) <= 50
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


# ------------------------------------------------ grouped Chebyshev products ----------------------------------------
@pytest.mark.parametrize("N,n_jobs,G", [(1, 1, 148), (40, 1, 148), (256, 1, 148), (256, 8, 148), (500, 2, 148),
                                        (1000, 4, 148), (2000, 1, 148), (2000, 8, 148), (4000, 3, 132), (1283, 16, 7)])
def test_grouped_work_list_covers_every_unit_of_every_job_once(N, n_jobs, G):
    """bml_symm_work_item: every (job, tile, k-slab) is covered exactly once; a split tile has one owner (the part that
    starts at k-slab 0) followed by its contributors on the next CTAs; at most one contributed partial per CTA."""
    bt = 32 if N <= 512 else (64 if N <= 1024 else 128)
    T = (N + bt - 1) // bt
    KT = (N + 15) // 16
    cover = {}
    units = []
    for c in range(G):
        items = api.bml_symm_work_items(N, n_jobs, G, c)
        n_contrib = 0
        for job, I, J, k0, k1, edge in items:
            assert edge == bt and 0 <= job < n_jobs and 0 <= I <= J < T and 0 <= k0 < k1 <= KT
            cover.setdefault((job, I, J), []).append((k0, k1, c))
            n_contrib += k0 > 0
        assert n_contrib <= 1
        units.append(sum(k1 - k0 for *_, k0, k1, _ in items))
    assert len(cover) == n_jobs * T * (T + 1) // 2
    W = (n_jobs * T * (T + 1) // 2) // G
    for parts in cover.values():
        parts.sort()
        assert parts[0][0] == 0 and parts[-1][1] == KT
        for (a0, a1, ca), (b0, b1, cb) in zip(parts, parts[1:]):
            assert a1 == b0 and cb > ca
        # the CTAs between the owner and its last contributor that hold no part of this tile have no part of the split
        # wave at all (fewer k-slabs than CTAs): the owner's scan skips them
        holders = [p[2] for p in parts]
        for cc in range(holders[0], holders[-1] + 1):
            assert cc in holders or units[cc] == W * KT
    assert sum(units) == n_jobs * T * (T + 1) // 2 * KT
    # the last, partial wave: either split along K evenly over all CTAs, or -- when the hand-off would cost more than
    # it saves (R KT / G + hs >= KT, hs = 2 / 8 / 20 slabs for tile edge 128 / 64 / 32) -- whole tiles on the first CTAs
    tail = [u - W * KT for u in units]
    R = n_jobs * T * (T + 1) // 2 - W * G
    hs = {128: 2, 64: 8, 32: 20}[bt]
    if R * KT + hs * G >= KT * G:
        assert tail == [KT] * R + [0] * (G - R)
        assert all(len(p) == 1 for p in cover.values()), "no tile is split"
    else:
        assert max(tail) - min(tail) <= 1


@pytest.mark.parametrize("k", list(range(2, 33)))
def test_doubling_schedule(k):
    """bml_cheb_schedule (reading C5): T_i = 2 T_a T_b - T_{a-b} with a + b = i, a - b in {0, 1}, and both operands
    come from strictly earlier levels (so one level is one grouped launch)."""
    sched = api.bml_cheb_schedule(k)
    assert [s[0] for s in sched] == list(range(2, k + 1))
    level_of = {0: 0, 1: 0}
    for i, lv, a, b in sched:
        assert a + b == i and a - b in (0, 1)
        assert level_of[a] < lv and level_of[b] < lv
        assert 2 ** (lv - 1) < i <= 2 ** lv
        level_of[i] = lv
    per_level = {}
    for i, lv, a, b in sched:
        per_level[lv] = per_level.get(lv, 0) + 1
    assert max(per_level.values()) <= api.SYMM_MAX_JOBS


def test_schedule_rejects_bad_k():
    L = api.load()
    assert L.bml_cheb_schedule(1, None, None, None) == -1
    assert L.bml_cheb_schedule(33, None, None, None) == -1
    assert L.bml_cheb_schedule(16, None, None, None) == 4


@pytest.mark.parametrize("sizes,G", [([5600, 5600, 5600, 5600], 148), ([896, 896, 896], 148), ([5657, 5810, 300, 1, 129], 148),
                                     ([200], 148), ([1500, 64], 7), ([128] * 40, 148), ([3000, 2000, 1000], 1)])
def test_batched_work_list_covers_every_unit_of_every_part_once(sizes, G):
    """The batched symmetric-square kernel of the graph-based SP2 solver (dense_batch.cu) over parts of UNEQUAL sizes:
    every CTA first takes W = tiles // G whole tiles dealt in waves (tile w G + c: concurrently running CTAs sit on
    consecutive tiles and share row panels in L2), then the units (16-column k-slabs) of the remaining tiles are cut
    into G equal contiguous ranges.  Every unit exactly once; a cut tile has one owner (the piece starting at k-slab 0)
    followed by contributors on the next CTAs; a CTA contributes to at most one tile and that piece is the FIRST item of
    its tail range (so hand-offs cannot cycle); only the last item of a range may be cut short."""
    tiles_of = [((n + 127) // 128) * ((n + 127) // 128 + 1) // 2 for n in sizes]
    W = sum(tiles_of) // G
    cover = {}
    tail_units = []
    for c in range(G):
        items = api.bml_dense_batch_work_items(sizes, G, c)
        assert len(items) >= W
        tail_units.append(sum(k1 - k0 for _, _, k0, k1, _ in items[W:]))
        flat0 = None
        for pos, (job, tile, k0, k1, KT) in enumerate(items):
            T = (sizes[job] + 127) // 128
            assert 0 <= job < len(sizes) and 0 <= tile < T * (T + 1) // 2 and KT == (sizes[job] + 15) // 16
            assert 0 <= k0 < k1 <= KT
            if pos < W:
                assert (k0, k1) == (0, KT)
                assert sum(tiles_of[:job]) + tile == pos * G + c, "wave w deals tile w G + c to CTA c"
            if k0 > 0:
                assert pos == W, "a contributed piece must come first in the CTA's tail range"
            if k1 < KT:
                assert pos == len(items) - 1, "only the last item of a range may be cut short"
            cover.setdefault((job, tile), []).append((k0, k1, c))
    want = {(j, t) for j, n in enumerate(sizes) for t in range(tiles_of[j])}
    assert set(cover) == want
    for (job, tile), parts in cover.items():
        KT = (sizes[job] + 15) // 16
        parts.sort()
        assert parts[0][0] == 0 and parts[-1][1] == KT
        for (a0, a1, ca), (b0, b1, cb) in zip(parts, parts[1:]):
            assert a1 == b0 and cb > ca
        # contributors are consecutive CTAs, up to CTAs whose tail range is empty (tiny batches on many CTAs)
        ctas = [p[2] for p in parts]
        assert all(tail_units[c] == 0 for c in range(ctas[0], ctas[-1] + 1) if c not in ctas)
    assert max(tail_units) - min(tail_units) <= 1
