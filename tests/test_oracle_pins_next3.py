"""Pins of the team collectives of the CPU oracle (NEXT-3): numpy on the member rows (concatenate, transpose, tile,
ufunc.reduce), the world team reproducing the world routines, non-members untouched, hand cases.  CPU only."""
import numpy as np
import pytest

from oracle import oracle as orc
from workloads import gen

TEAMS = [(0, 1, 8), (1, 2, 4), (2, 3, 2), (5, 1, 3), (7, 1, 1), (0, 7, 2)]


def filled(npes, nbytes, seed):
    w = orc.OracleWorld(npes, 3 * nbytes + 1024)
    s, d = w.malloc(nbytes), w.malloc(nbytes)
    pay = gen.u64(npes * (nbytes // 8), seed).view(np.uint8).reshape(npes, nbytes)
    w.view(s, nbytes)[:] = pay
    w.view(d, nbytes)[:] = 0xEE
    return w, s, d, pay


def members(team):
    return [team[0] + k * team[1] for k in range(team[2])]


@pytest.mark.parametrize("team", TEAMS)
def test_team_fcollect_alltoall_broadcast_equal_numpy_on_member_rows(team):
    npes, blk = 8, 40
    m = members(team)
    out = [p for p in range(npes) if p not in m]
    w, s, d, pay = filled(npes, blk * 8, 501)
    w.team_fcollect(team, d, s, blk)
    assert np.array_equal(w.view(d, blk * 8)[m, :blk * len(m)], np.tile(np.concatenate([pay[p, :blk] for p in m]), (len(m), 1)))
    assert (w.view(d, blk * 8)[out] == 0xEE).all() and (w.view(d, blk * 8)[m, blk * len(m):] == 0xEE).all()
    w, s, d, pay = filled(npes, blk * 8, 502)
    w.team_alltoall(team, d, s, blk)
    src = pay[m, :blk * len(m)].reshape(len(m), len(m), blk)
    assert np.array_equal(w.view(d, blk * 8)[m, :blk * len(m)].reshape(len(m), len(m), blk), src.transpose(1, 0, 2))
    assert (w.view(d, blk * 8)[out] == 0xEE).all()
    w, s, d, pay = filled(npes, blk * 8, 503)
    root = len(m) - 1
    w.team_broadcast(team, d + 3, s + 5, 100, root)
    assert np.array_equal(w.view(d, blk * 8)[m, 3:103], np.tile(pay[m[root], 5:105], (len(m), 1)))
    assert (w.view(d, blk * 8)[out] == 0xEE).all() and np.array_equal(w.view(s, blk * 8), pay)


@pytest.mark.parametrize("team", TEAMS)
@pytest.mark.parametrize("op,uf", [("sum", np.add), ("max", np.maximum), ("xor", np.bitwise_xor)])
def test_team_reduce_equals_ufunc_reduce_over_member_rows(team, op, uf):
    npes, n = 8, 33
    m = members(team)
    w, s, d, pay = filled(npes, n * 8, 504)
    w.team_reduce(team, op, "i64", d, s, n)
    exp = uf.reduce(pay.view(np.int64)[m], axis=0)
    assert np.array_equal(w.view(d, n * 8, np.int64)[m], np.tile(exp, (len(m), 1)))
    out = [p for p in range(npes) if p not in m]
    assert (w.view(d, n * 8)[out] == 0xEE).all()


def test_world_team_reproduces_the_world_routines_and_bad_teams_are_rejected():
    npes, blk = 6, 24
    for name, args in (("fcollect", (blk,)), ("alltoall", (blk,)), ("broadcast", (blk, 4))):
        w1, s, d, _ = filled(npes, blk * 8, 505)
        w2, _, _, _ = filled(npes, blk * 8, 505)
        getattr(w1, "team_" + name)((0, 1, npes), d, s, *args)
        getattr(w2, name)(d, s, *args)
        assert np.array_equal(w1.heap, w2.heap), name
    w1, s, d, _ = filled(npes, blk * 8, 506)
    w2, _, _, _ = filled(npes, blk * 8, 506)
    f = gen.normal_f32(npes * blk, 507).reshape(npes, blk)
    w1.view(s, blk * 4, np.float32)[:] = f
    w2.view(s, blk * 4, np.float32)[:] = f
    w1.team_reduce((0, 1, npes), "sum", "f32", d, s, blk)
    w2.sum_reduce_f32(d, s, blk)
    assert np.array_equal(w1.heap, w2.heap)
    for bad in ((0, 1, 7), (4, 2, 2), (-1, 1, 2), (0, 0, 2), (0, 1, 0)):
        with pytest.raises(orc.OracleError):
            w1.team_fcollect(bad, d, s, 8)
    with pytest.raises(orc.OracleError):
        w1.team_broadcast((1, 2, 2), d, s, 8, 2)                     # root is a team rank


def test_team_hand_case():
    w = orc.OracleWorld(4, 64)
    w.heap[:, :2] = [[1, 2], [3, 4], [5, 6], [7, 8]]
    w.team_alltoall((1, 2, 2), 8, 0, 1)                              # members: PE 1 (rank 0), PE 3 (rank 1)
    assert w.heap[:, 8:10].tolist() == [[0, 0], [3, 7], [0, 0], [4, 8]]
    w.team_fcollect((0, 3, 2), 16, 0, 2)                             # members: PE 0, PE 3
    assert w.heap[:, 16:20].tolist() == [[1, 2, 7, 8], [0, 0, 0, 0], [0, 0, 0, 0], [1, 2, 7, 8]]
