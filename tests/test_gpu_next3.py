"""GPU parity of the team collectives (NEXT-3) against the CPU oracle, through the C-ABI: strided teams, nested splits,
single-member teams, the world team; bulk and any-alignment paths; non-members must stay untouched."""
import numpy as np
import pytest
import torch

from oracle import oracle as orc
from paper_2607_08006_b200 import World
from paper_2607_08006_b200.binding import F32, I64, RED, TEAM, ShmemgError
from workloads import gen

pytestmark = pytest.mark.gpu
DEV = "cuda:0"
TEAMS = [(0, 1, 12), (1, 2, 5), (2, 3, 4), (5, 1, 3), (11, 1, 1), (0, 11, 2)]


def setup(npes, nbytes, seed):
    hb = 3 * nbytes + 4096
    w, ow = World(npes, hb, DEV), orc.OracleWorld(npes, hb)
    s, d = w.malloc(nbytes), w.malloc(nbytes)
    os_, od = ow.malloc(nbytes), ow.malloc(nbytes)
    pay = gen.u64(npes * (nbytes // 8), seed).view(np.uint8).reshape(npes, nbytes)
    w.view(s, nbytes).copy_(torch.from_numpy(pay)); ow.view(os_, nbytes)[:] = pay
    w.view(d, nbytes).fill_(0xEE); ow.view(od, nbytes)[:] = 0xEE
    return w, ow, s, d, os_, od


def same(w, ow, off, ooff, nbytes):
    return np.array_equal(w.view(off, nbytes).cpu().numpy(), ow.view(ooff, nbytes))


@pytest.mark.parametrize("team", TEAMS)
@pytest.mark.parametrize("blk,shift", [(40000, 0), (4099, 3)])
def test_team_collectives_match_oracle(team, blk, shift):
    npes = 12
    nbytes = (blk * 12 + 64 + 255) // 256 * 256
    w, ow, s, d, os_, od = setup(npes, nbytes, 601)
    t = w.team_split_strided(TEAM.WORLD, *team)
    assert w.team_n_pes(t) == team[2] and w.team_translate_pe(t, team[2] - 1) == team[0] + (team[2] - 1) * team[1]
    b16 = blk // 16 * 16 if shift == 0 else blk
    w.team_fcollect(t, d + shift, s + shift, b16); ow.team_fcollect(team, od + shift, os_ + shift, b16)
    w.quiet(0)
    assert same(w, ow, d, od, nbytes)
    w.view(d, nbytes).fill_(0xEE); ow.view(od, nbytes)[:] = 0xEE
    w.team_alltoall(t, d + shift, s + shift, b16); ow.team_alltoall(team, od + shift, os_ + shift, b16)
    w.quiet(0)
    assert same(w, ow, d, od, nbytes)
    w.view(d, nbytes).fill_(0xEE); ow.view(od, nbytes)[:] = 0xEE
    root = team[2] // 2
    w.team_broadcast(t, d + shift, s + shift, b16, root); ow.team_broadcast(team, od + shift, os_ + shift, b16, root)
    w.quiet(0)
    assert same(w, ow, d, od, nbytes) and same(w, ow, s, os_, nbytes)


@pytest.mark.parametrize("team", TEAMS)
@pytest.mark.parametrize("op,oname,dtype,dname,es", [(RED.SUM, "sum", I64, "i64", 8), (RED.MAX, "max", I64, "i64", 8),
                                                      (RED.XOR, "xor", I64, "i64", 8), (RED.SUM, "sum", F32, "f32", 4)])
def test_team_reduce_matches_oracle(team, op, oname, dtype, dname, es):
    npes, n = 12, 30011
    nbytes = (n * 8 + 255) // 256 * 256
    w, ow, s, d, os_, od = setup(npes, nbytes, 602)
    if dtype == F32:
        f = gen.normal_f32(npes * n, 603).reshape(npes, n)
        w.view(s, n * 4, torch.float32).copy_(torch.from_numpy(f)); ow.view(os_, n * 4, np.float32)[:] = f
    t = w.team_split_strided(TEAM.WORLD, *team)
    w.team_reduce(t, op, dtype, d, s, n); ow.team_reduce(team, oname, dname, od, os_, n)
    w.quiet(0)
    assert same(w, ow, d, od, nbytes) and same(w, ow, s, os_, nbytes)


def test_nested_split_world_team_and_errors():
    npes, blk = 16, 4096
    w, ow, s, d, os_, od = setup(npes, blk * 16, 604)
    even = w.team_split_strided(TEAM.WORLD, 0, 2, 8)                 # PEs 0,2,..,14
    sub = w.team_split_strided(even, 1, 3, 3)                        # ranks 1,4,7 of `even` = PEs 2, 8, 14
    assert [w.team_translate_pe(sub, k) for k in range(3)] == [2, 8, 14]
    w.team_alltoall(sub, d, s, blk); ow.team_alltoall((2, 6, 3), od, os_, blk)
    w.team_fcollect(TEAM.DEVICE_WORLD, d + 3 * blk * 0, s, 0)        # zero-size on a predefined team: no-op
    w.quiet(0)
    assert same(w, ow, d, od, blk * 16)
    w.team_fcollect(TEAM.WORLD, d, s, blk); ow.fcollect(od, os_, blk)  # the world team = the world collective
    w.quiet(0)
    assert same(w, ow, d, od, blk * 16)
    assert w.query_capabilities(sub) == w.query_capabilities(TEAM.WORLD)
    for bad in ((0, 1, 17), (8, 2, 5), (-1, 1, 2), (0, 0, 2), (0, 1, 0)):
        with pytest.raises(ShmemgError):
            w.team_split_strided(TEAM.WORLD, *bad)
    with pytest.raises(ShmemgError):
        w.team_split_strided(even, 0, 1, 9)                          # larger than the parent
    with pytest.raises(ShmemgError):
        w.team_broadcast(sub, d, s, 64, 3)                           # root is a team rank
    with pytest.raises(ShmemgError):
        w.team_fcollect(99, d, s, 64)
    w.put(d, s, 64, 15, 0); w.quiet(0)                               # the world is intact after team calls
    assert w.npes == 16
