"""Degenerate cases of the hot path on the GPU against the oracle: a single PE (every collective degenerates to a copy or the
identity), zero-length calls, a transfer that fills the whole heap window, an AMO batch where every op hits one word."""
import numpy as np
import pytest
import torch

from oracle import oracle as orc
from paper_2607_08006_b200 import World
from paper_2607_08006_b200.binding import AMO, AMO_HOT_AGGREGATE, F32, I64, RED
from workloads import gen

pytestmark = pytest.mark.gpu
DEV = "cuda:0"


def test_single_pe_world_collectives_degenerate_to_copies():
    nb = 70000 * 8
    w, ow = World(1, 3 * nb + 4096, DEV), orc.OracleWorld(1, 3 * nb + 4096)
    s, d = w.malloc(nb), w.malloc(nb)
    os_, od = ow.malloc(nb), ow.malloc(nb)
    x = gen.u64(nb // 8, 401).reshape(1, -1)
    w.view(s, nb, torch.int64).copy_(torch.from_numpy(x.view(np.int64)))
    ow.view(os_, nb, np.uint64)[:] = x
    for name, g, o in (("alltoall", lambda: w.alltoall(d, s, nb), lambda: ow.alltoall(od, os_, nb)),
                       ("fcollect", lambda: w.fcollect(d, s, nb), lambda: ow.fcollect(od, os_, nb)),
                       ("broadcast", lambda: w.broadcast(d, s, nb, 0), lambda: ow.broadcast(od, os_, nb, 0)),
                       ("sum_i64", lambda: w.sum_reduce(I64, d, s, nb // 8), lambda: ow.sum_reduce_i64(od, os_, nb // 8)),
                       ("max_i64", lambda: w.reduce(RED.MAX, I64, d, s, nb // 8), lambda: ow.reduce("max", "i64", od, os_, nb // 8)),
                       ("sum_f32", lambda: w.reduce(RED.MIN, F32, d, s, 1000), lambda: ow.reduce("min", "f32", od, os_, 1000))):
        if name == "sum_f32":                            # finite fp32 inputs for the float case
            f = gen.normal_f32(1000, 402).reshape(1, -1)
            w.view(s, 4000, torch.float32).copy_(torch.from_numpy(f)); ow.view(os_, 4000, np.float32)[:] = f
        w.view(d, nb).zero_(); ow.view(od, nb)[:] = 0
        g(); w.quiet(0); o()
        assert np.array_equal(w.view(d, nb).cpu().numpy(), ow.view(od, nb)), name
    w.barrier_all(); w.barrier_all_repeat(5)
    w.put(d, s, nb, 0, 0); w.quiet(0)                     # a put to oneself
    assert np.array_equal(w.view(d, nb).cpu().numpy(), w.view(s, nb).cpu().numpy())


def test_zero_length_calls_are_no_ops():
    w = World(3, 1 << 16, DEV)
    a, b = w.malloc(4096), w.malloc(4096)
    w.view(a, 4096).fill_(7); w.view(b, 4096).fill_(9)
    e32 = torch.empty(0, dtype=torch.int32, device=DEV)
    e64 = torch.empty(0, dtype=torch.int64, device=DEV)
    w.alltoall(b, a, 0); w.fcollect(b, a, 0); w.broadcast(b, a, 0, 1); w.sum_reduce(I64, b, a, 0); w.reduce(RED.XOR, I64, b, a, 0)
    w.put(b, a, 0, 0, 1); w.get(b, a, 0, 2, 1); w.ibput(b, a, 8, 8, 8, 0, 0, 1); w.ibget(b, a, 8, 8, 0, 5, 0, 1)
    w.atomic_add_batch(a, e32, e32, val_scalar=1); w.atomic_fetch_add_batch(a, e32, e32, e64, val_scalar=1, flags=AMO_HOT_AGGREGATE)
    w.atomic_compare_swap_batch(a, e32, e32, e64, cond_scalar=0, val_scalar=1)
    w.atomic_op_batch(AMO.SWAP, 8, a, e32, e32, val_scalar=3, fetched_out=e64)
    w.quiet(0)
    assert (w.view(a, 4096).cpu().numpy() == 7).all() and (w.view(b, 4096).cpu().numpy() == 9).all()


def test_whole_window_transfer_and_single_word_storm():
    hb = 3 << 20
    w, ow = World(2, hb, DEV), orc.OracleWorld(2, hb)
    pay = gen.u64(2 * hb // 8, 403).view(np.uint8).reshape(2, hb)
    w.view(0, hb).copy_(torch.from_numpy(pay)); ow.view(0, hb)[:] = pay
    w.put(0, 0, hb, 0, 1); w.quiet(0)                     # PE 0's whole window over PE 1's
    ow.heap[1, :] = ow.heap[0, :]
    assert np.array_equal(w.view(0, hb).cpu().numpy(), ow.view(0, hb))
    # 2^21 fetch-adds on ONE word (every op hot), hot-set aggregation on: fetched values are exactly 0..n-1 times the value
    n = 1 << 21
    w.view(0, 8, torch.int64).zero_()
    z = torch.zeros(n, dtype=torch.int32, device=DEV)
    f = torch.empty(n, dtype=torch.int64, device=DEV)
    w.set_scratch_for(n)
    w.atomic_fetch_add_batch(0, z, z, f, val_scalar=3, flags=AMO_HOT_AGGREGATE)
    w.quiet(0)
    assert w.view(0, 8, torch.int64).cpu().numpy()[0, 0] == 3 * n
    assert np.array_equal(np.sort(f.cpu().numpy()), 3 * np.arange(n, dtype=np.int64))


def test_realign_counters_after_short_participation():
    """A kernel that left its barrier round unfinished (here: three stray arrivals written straight into the control region, as an
    aborted kernel would leave them) makes the round arithmetic of every later in-kernel barrier wrong.  After
    shmemg_realign_counters_on_stream the stamped barrier invariant holds again; on an intact world the call changes nothing."""
    npes = 8
    w = World(npes, 4096, DEV)
    st = w.calloc(3, 8)
    w.barrier_all_repeat(50, st)
    w.realign_counters()                                     # nothing wrong: no change
    w.quiet(0)
    ctl = w.slab[npes * w.stride:].view(torch.int64)         # control region: [0] barrier epoch, [1] in-kernel arrivals
    assert int(ctl[1]) == 50 * npes
    ctl[1] += 3                                              # residue of an unfinished round
    w.realign_counters()
    w.quiet(0)
    assert int(ctl[1]) == 51 * npes
    w.view(st, 24, torch.int64).zero_()
    w.barrier_all_repeat(1000, st)
    w.quiet(0)
    sv = w.view(st, 24, torch.int64).cpu().numpy()
    assert (sv[:, 2] == 0).all() and int(ctl[1]) == 1051 * npes
    # the sampling kernel's arrival counter (16 CTAs per call) is realigned the same way
    n = 1 << 20
    a = w.calloc(8, 8)
    z = torch.zeros(n, dtype=torch.int32, device=DEV)
    f = torch.empty(n, dtype=torch.int64, device=DEV)
    w.set_scratch_for(n)
    hot_done = w.slab[npes * w.stride:].view(torch.int32)
    off = (16 + 48 + 4 * 1024 + 4 * 128 + 4 + 4 + 8 + 4) // 4                # offsetof(CtlRegion, hot_done) / 4
    w.atomic_fetch_add_batch(a, z, z, f, val_scalar=1, flags=AMO_HOT_AGGREGATE)
    w.quiet(0)
    assert int(hot_done[off]) == 16
    hot_done[off] += 5
    w.realign_counters()
    w.atomic_fetch_add_batch(a, z, z, f, val_scalar=1, flags=AMO_HOT_AGGREGATE)
    w.quiet(0)
    assert int(hot_done[off]) == 48
    assert np.array_equal(np.sort(f.cpu().numpy()), np.arange(n, 2 * n))
