"""Pins of the oracle's PE -> GPU placement (NEXT-4 (iii); SURVEY 8(e) "PE p -> GPU p mod G", reading 42).

The sharded operations add no arithmetic: a sharded world computes what ONE world of all the PEs computes, so their oracle is
the existing routine on the global world.  What is new is WHERE a PE's window lives; that placement is pinned here against
things other than itself: a hand-written table, the bijection property by brute force, numpy strided slicing of the global
heap, and the closed form of a sharded alltoall."""
import numpy as np
import pytest

from oracle import oracle as orc


def test_placement_hand_table_two_shards_eight_pes():
    # global PE:            0  1  2  3  4  5  6  7
    assert [orc.shard_of(g, 2) for g in range(8)] == [0, 1, 0, 1, 0, 1, 0, 1]
    assert [orc.shard_local_index(g, 2) for g in range(8)] == [0, 0, 1, 1, 2, 2, 3, 3]
    # three shards, seven PEs (ragged: shard 0 holds three PEs, the others two)
    assert [orc.shard_of(g, 3) for g in range(7)] == [0, 1, 2, 0, 1, 2, 0]
    assert [orc.shard_local_index(g, 3) for g in range(7)] == [0, 0, 0, 1, 1, 1, 2]


@pytest.mark.parametrize("G", [1, 2, 3, 4, 8, 16])
def test_placement_is_a_bijection(G):
    n = 5 * G + 3
    seen = set()
    for g in range(n):
        s, l = orc.shard_of(g, G), orc.shard_local_index(g, G)
        assert 0 <= s < G and l >= 0
        assert orc.shard_global_pe(s, l, G) == g              # inverse
        assert (s, l) not in seen                             # injective
        seen.add((s, l))
    # dense: shard s holds local indices 0 .. count-1 with no hole
    for s in range(G):
        ls = sorted(l for (ss, l) in seen if ss == s)
        assert ls == list(range(len(ls)))
    # one shard is the unsharded world
    if G == 1:
        assert all(orc.shard_local_index(g, 1) == g for g in range(n))


@pytest.mark.parametrize("G,npes", [(2, 8), (4, 8), (3, 9), (1, 5)])
def test_shard_rows_are_a_strided_slice_of_the_global_heap(G, npes):
    ow = orc.OracleWorld(npes, 4096)
    off = ow.malloc(1024)
    rng = np.random.default_rng(7)
    ow.view(off, 1024)[:] = rng.integers(0, 256, (npes, 1024), dtype=np.uint8)
    for s in range(G):
        assert np.array_equal(orc.shard_rows(ow, s, G, off, 1024), ow.view(off, 1024)[s::G])       # numpy's own strided slice
    # the shards partition the heap: stacking them back in (local, shard) order gives the global rows
    if npes % G == 0:
        stacked = np.stack([orc.shard_rows(ow, s, G, off, 1024) for s in range(G)], axis=1).reshape(npes, 1024)
        assert np.array_equal(stacked, ow.view(off, 1024))


def test_sharded_alltoall_closed_form():
    """alltoall on the global world, seen shard by shard: the block that local PE l of shard s receives from global PE j is
    block g = l*G + s of j's source -- the transpose identity with the placement substituted."""
    G, L, blk = 2, 3, 64
    npes = G * L
    ow = orc.OracleWorld(npes, 2 * npes * blk + 512)
    src, dst = ow.malloc(npes * blk), ow.malloc(npes * blk)
    rng = np.random.default_rng(11)
    S = rng.integers(0, 256, (npes, npes, blk), dtype=np.uint8)
    ow.view(src, npes * blk)[:] = S.reshape(npes, -1)
    ow.alltoall(dst, src, blk)
    for s in range(G):
        rows = orc.shard_rows(ow, s, G, dst, npes * blk).reshape(-1, npes, blk)
        for l in range(rows.shape[0]):
            g = orc.shard_global_pe(s, l, G)
            for j in range(npes):
                assert np.array_equal(rows[l, j], S[j, g])
