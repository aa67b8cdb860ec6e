"""GPU parity on the five BASELINE configs and the single-op / collective entry points,
through the C-ABI, against the CPU oracle.  Bit-exact for copies and integer atomics; fp32 sum_reduce
within 1e-6 relative (+2^-36 absolute floor, reading 14) of the fp64 oracle."""
import numpy as np
import pytest
import torch

from gpu_common import DEV, assert_objects_equal, heap_bytes_for, run_gpu, run_oracle, to_dev
from invariants import check_compare_swap_claim, check_fetch_add
from oracle import oracle as orc
from paper_2607_08006_b200 import CAP, CMP, ERR, SIGNAL, TEAM, ShmemgError, World
from paper_2607_08006_b200.binding import (AMO_HOT_AGGREGATE, AMO_TEST_BEFORE_SWAP, AMO_THEN_BARRIER, AMO_WARP_AGGREGATE,
                                           F32, I64)
from paper_2607_08006_b200.loader import Loaded
from workloads import configs, gen

pytestmark = pytest.mark.gpu
M64 = (1 << 64) - 1


# ---- a1-a4: heap, allocator, translation, capabilities -----------------------------------------------------
def test_world_allocator_translation_capabilities():
    w = World(5, 1 << 20, DEV)
    caps = w.query_capabilities(TEAM.WORLD)
    for bit in (CAP.GPU_HEAP_PRESENT, CAP.DEFAULT_HEAP_IS_GPU, CAP.HOST_INITIATED_GPU_BUFFERS, CAP.STREAM_TRIGGERED,
                CAP.PTR_DEVICE_ACCESSIBLE, CAP.PROGRESS_GPU_ONLY, CAP.PATH_DIRECT):
        assert caps & bit
    assert not caps & CAP.PTR_HOST_ACCESSIBLE and not caps & CAP.DEVICE_COLLECTIVES
    assert w.query_capabilities(TEAM.DEVICE_WORLD) & CAP.DEVICE_INITIATED
    with pytest.raises(ShmemgError):
        w.query_capabilities(17)
    a, b = w.malloc(1000), w.malloc(1)
    assert a % 256 == 0 and b % 256 == 0 and b >= a + 1000
    c = w.align(65536, 100)
    assert c % 65536 == 0
    # space symmetry: the same offset addresses a valid, disjoint window on every PE
    base = w.slab.data_ptr()
    ptrs = [w.ptr(a, p) for p in range(5)]
    assert ptrs == [base + p * w.stride + a for p in range(5)]
    assert w.ptr(a, 5) == 0 and w.ptr(1 << 20, 0) == 0
    w.free(b)
    assert w.malloc(200) == b                         # first fit reuses the freed block
    w.free(a)
    with pytest.raises(ShmemgError):
        w.free(a)
    with pytest.raises(ShmemgError) as e:
        w.malloc(1 << 21)
    assert e.value.code == ERR.NOMEM
    w.view(c, 256).fill_(0xAB)
    z = w.calloc(32, 8)
    assert z != c and (w.view(z, 256).cpu().numpy() == 0).all()
    # writes through one PE's pointer land in that PE's window only
    w.view(z, 256)[3].fill_(7)
    v = w.view(z, 256).cpu().numpy()
    assert (v[3] == 7).all() and (np.delete(v, 3, axis=0) == 0).all()


# ---- a6-a8: single ops on a stream -----------------------------------------------------------------------------
def test_single_put_get_put_signal_wait_on_stream():
    npes, nb = 4, 3 << 20
    w = World(npes, 4 * nb, DEV)
    ow = orc.OracleWorld(npes, 4 * nb)
    s, d, sig = w.malloc(nb), w.malloc(nb), w.calloc(8, 8)
    os_, od, osig = ow.malloc(nb), ow.malloc(nb), ow.malloc(64)
    pay = gen.u64(npes * nb // 8, 31).view(np.uint8).reshape(npes, nb)
    w.view(s, nb).copy_(torch.from_numpy(pay))
    w.view(d, nb).zero_()
    ow.view(os_, nb)[:] = pay
    cases = [(0, 0, nb, 0, 1), (3, 5, 1000001, 1, 2), (16, 16, 1 << 20, 2, 3), (7, 2, 13, 3, 0), (1, 1, 0, 0, 2)]
    from workloads.spec import Program
    for k, (so, do, n, pe, tgt) in enumerate(cases):
        if k % 2 == 0:
            w.put(d + do, s + so, n, pe, tgt)
            ow.heap[tgt, od + do:od + do + n] = ow.heap[pe, os_ + so:os_ + so + n]
        else:
            w.get(d + do, s + so, n, pe, tgt)
            ow.heap[pe, od + do:od + do + n] = ow.heap[tgt, os_ + so:os_ + so + n]
    # put_signal then a stream-level wait that is already satisfiable by the earlier op
    w.put_signal(d + 64, s + 128, 2 << 20, sig + 8, 41, SIGNAL.SET, 1, 3)
    w.put_signal(d + 64, s + 128, 0, sig + 8, 1, SIGNAL.ADD, 2, 3)
    w.signal_wait_until(sig + 8, CMP.EQ, 42, 3)
    w.fence(0)
    w.quiet_on_stream(1)
    w.quiet(3)
    ow.heap[3, od + 64:od + 64 + (2 << 20)] = ow.heap[1, os_ + 128:os_ + 128 + (2 << 20)]
    assert np.array_equal(w.view(d, nb).cpu().numpy(), ow.view(od, nb))
    assert w.view(sig, 64, torch.int64).cpu().numpy()[3, 1] == 42
    with pytest.raises(ShmemgError):
        w.put(d, s, 4 * nb, 0, 1)               # runs past the end of the heap window
    with pytest.raises(ShmemgError):
        w.put_signal(d, s, 8, sig + 4, 1, SIGNAL.SET, 0, 1)


# ---- C1 ---------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("flags", [0, AMO_WARP_AGGREGATE])
@pytest.mark.parametrize("idx_dtype", [np.int64, np.int32])
def test_c1_atomic_add_bit_exact(flags, idx_dtype):
    wl = configs.c1_atomic_add()
    w = World(wl.npes, wl.nelem * 8 + 4096, DEV)
    a = w.calloc(wl.nelem, 8)
    w.atomic_add_batch(a, to_dev(wl.tgt_pe), to_dev(wl.idx.astype(idx_dtype)), val=to_dev(wl.val), flags=flags)
    w.quiet(0)                      # quiet + barrier as config 1 prescribes
    w.barrier_all()
    ow = orc.OracleWorld(wl.npes, wl.nelem * 8 + 4096)
    oa = ow.malloc(wl.nelem * 8)
    ow.atomic_add_batch(oa, wl.tgt_pe, wl.idx, wl.val)
    assert np.array_equal(w.view(a, wl.nelem * 8).cpu().numpy(), ow.view(oa, wl.nelem * 8))


def test_c1_quiet_and_barrier_folded_into_the_amo_launch():
    """SHMEMG_AMO_THEN_BARRIER: one launch does the adds, the quiet and the barrier (epoch bump by the last CTA); every AMO
    entry point, the hot-set kernels and the empty call included."""
    wl = configs.c1_atomic_add()
    w = World(wl.npes, wl.nelem * 8 + 4096, DEV)
    a = w.calloc(wl.nelem, 8)
    t, i, v = to_dev(wl.tgt_pe), to_dev(wl.idx.astype(np.int64)), to_dev(wl.val)
    e0, l0 = w.barrier_epoch(), w.launches
    w.atomic_add_batch(a, t, i, val=v, flags=AMO_THEN_BARRIER)
    assert w.launches == l0 + 1 and w.barrier_epoch() == e0 + 1
    ow = orc.OracleWorld(wl.npes, wl.nelem * 8 + 4096)
    oa = ow.malloc(wl.nelem * 8)
    ow.atomic_add_batch(oa, wl.tgt_pe, wl.idx, wl.val)
    assert np.array_equal(w.view(a, wl.nelem * 8).cpu().numpy(), ow.view(oa, wl.nelem * 8))
    f = torch.empty(len(wl.val), dtype=torch.int64, device=DEV)
    w.atomic_fetch_add_batch(a, t, i, f, val=v, flags=AMO_THEN_BARRIER)
    w.atomic_compare_swap_batch(a, t, i, f, cond_scalar=0, val_scalar=1, flags=AMO_THEN_BARRIER)
    e = torch.empty(0, dtype=torch.int32, device=DEV)
    w.atomic_add_batch(a, e, e, val_scalar=1, flags=AMO_THEN_BARRIER)                # no ops: still a barrier
    assert w.barrier_epoch() == e0 + 4
    n = 1 << 20
    w.set_scratch_for(n)
    z = torch.zeros(n, dtype=torch.int32, device=DEV)
    f = torch.empty(n, dtype=torch.int64, device=DEV)
    w.atomic_fetch_add_batch(a, z, z, f, val_scalar=1, flags=AMO_THEN_BARRIER | AMO_HOT_AGGREGATE)
    w.atomic_add_batch(a, z, z, val_scalar=1, flags=AMO_THEN_BARRIER | AMO_HOT_AGGREGATE)
    assert w.barrier_epoch() == e0 + 6


def test_atomic_add_heavy_contention_and_scalar_value():
    n = 1 << 20
    w = World(2, 4096, DEV)
    a = w.calloc(8, 8)
    tgt = torch.zeros(n, dtype=torch.int32, device=DEV)
    idx = (torch.arange(n, device=DEV) % 3).to(torch.int32)
    for flags in (0, AMO_WARP_AGGREGATE, AMO_HOT_AGGREGATE, AMO_HOT_AGGREGATE):
        w.atomic_add_batch(a, tgt, idx, val=None, val_scalar=M64, flags=flags)       # adds -1 (wraparound)
        w.set_scratch_for(n)                   # third pass: no scratch registered -> the plain kernel; fourth: the hot-set kernels
    w.quiet(0)
    v = w.view(a, 64, torch.int64).cpu().numpy()
    cnt = np.bincount(np.arange(n) % 3, minlength=3)
    assert v[0, :3].tolist() == (-4 * cnt).tolist() and v[1].sum() == 0


@pytest.mark.parametrize("n", [1, 1025, 3 * 8192 + 77, (1 << 20) + 5, (1 << 21) + 1029])
@pytest.mark.parametrize("flags", [0, AMO_WARP_AGGREGATE, AMO_HOT_AGGREGATE])
@pytest.mark.parametrize("idx_dtype", [np.int64, np.uint32])
def test_fetch_add_skewed_scalar_value_ragged(n, flags, idx_dtype):
    """Ragged sizes, a skewed key distribution (many duplicates inside one warp), a scalar value > 1, non-zero initial
    contents, an array that does not start at offset 0; per word the fetched values must be a permutation of the prefix
    sums and the final words bit-exact."""
    npes, words = 3, 5000
    w = World(npes, words * 8 + 8192, DEV)
    pad = w.malloc(256)                                      # the array does not start at offset 0
    a = w.malloc(words * 8)
    init = (gen.u64(npes * words, 77) >> np.uint64(2)).reshape(npes, words)
    w.view(a, words * 8, torch.int64).copy_(torch.from_numpy(init.view(np.int64)))
    r = gen.u64(n, 78)
    key = ((r % np.uint64(npes * words)) >> (r >> np.uint64(60))).astype(np.int64)      # skewed towards small keys
    tgt, idx = (key // words).astype(np.int32), (key % words).astype(idx_dtype)
    f = torch.empty(n, dtype=torch.int64, device=DEV)
    w.set_scratch_for(n)                                     # caller-owned scratch of the hot-set kernels
    w.atomic_fetch_add_batch(a, to_dev(tgt), to_dev(idx), f, val=None, val_scalar=7, flags=flags)
    w.quiet(0)
    fin = w.view(a, words * 8, torch.int64).cpu().numpy().view(np.uint64).reshape(-1)
    ow = orc.OracleWorld(npes, words * 8 + 8192)
    ow.malloc(256)
    oa = ow.malloc(words * 8)
    ow.view(oa, words * 8, np.uint64)[:] = init
    ow.atomic_fetch_add_batch(oa, tgt, idx.astype(np.int64), np.full(n, 7, dtype=np.uint64))
    assert np.array_equal(fin, ow.view(oa, words * 8, np.uint64).reshape(-1))           # final words bit-exact
    check_fetch_add(key, np.full(n, 7, dtype=np.uint64), f.cpu().numpy().view(np.uint64), init.reshape(-1), fin)


# ---- C4 ---------------------------------------------------------------------------------------------------------
def _run_c4(g, flags):
    vpp, E = g.verts_per_pe, len(g.u)
    w = World(g.npes, 2 * vpp * 8 + 4096, DEV)
    deg = w.calloc(vpp, 8)
    par = w.malloc(vpp * 8)
    w.view(par, vpp * 8, torch.int64).fill_(-1)
    f_deg = torch.empty(E, dtype=torch.int64, device=DEV)
    f_par = torch.empty(E, dtype=torch.int64, device=DEV)
    w.set_scratch_for(E)
    w.atomic_fetch_add_batch(deg, to_dev(g.owner(g.u)), to_dev(g.local(g.u).astype(np.uint32)), f_deg, val=None,
                             val_scalar=1, flags=flags)
    w.atomic_compare_swap_batch(par, to_dev(g.owner(g.v)), to_dev(g.local(g.v).astype(np.uint32)), f_par,
                                cond=None, cond_scalar=M64, val=to_dev(g.u.astype(np.uint64)), flags=flags)
    w.quiet(0)
    degs = w.view(deg, vpp * 8, torch.int64).cpu().numpy().view(np.uint64).reshape(-1)
    pars = w.view(par, vpp * 8, torch.int64).cpu().numpy().view(np.uint64).reshape(-1)
    return degs, pars, f_deg.cpu().numpy().view(np.uint64), f_par.cpu().numpy().view(np.uint64)


@pytest.mark.parametrize("flags", [0, AMO_WARP_AGGREGATE, AMO_TEST_BEFORE_SWAP, AMO_WARP_AGGREGATE | AMO_TEST_BEFORE_SWAP,
                                   AMO_HOT_AGGREGATE | AMO_TEST_BEFORE_SWAP])
def test_c4_graph_small_full_oracle(flags):
    g = configs.c4_graph(scale=16, edge_factor=16, npes=32)
    degs, pars, f_deg, f_par = _run_c4(g, flags)
    vpp, E = g.verts_per_pe, len(g.u)
    ow = orc.OracleWorld(g.npes, 2 * vpp * 8 + 512)
    od, op = ow.malloc(vpp * 8), ow.malloc(vpp * 8)
    ow.view(op, vpp * 8, np.uint64)[:] = M64
    ow.atomic_fetch_add_batch(od, g.owner(g.u), g.local(g.u), np.ones(E, dtype=np.uint64))
    ow.atomic_compare_swap_batch(op, g.owner(g.v), g.local(g.v), np.full(E, M64, dtype=np.uint64), g.u.astype(np.uint64))
    assert np.array_equal(degs, ow.view(od, vpp * 8, np.uint64).reshape(-1))          # degrees bit-exact
    # claimed-or-not is schedule independent; which in-neighbour won is not
    assert np.array_equal(pars == M64, ow.view(op, vpp * 8, np.uint64).reshape(-1) == M64)
    check_fetch_add(g.u.astype(np.int64), np.ones(E, dtype=np.uint64), f_deg, np.zeros(1 << g.scale, dtype=np.uint64), degs)
    check_compare_swap_claim(g.v.astype(np.int64), g.u.astype(np.uint64), f_par, pars)
    edges = (g.u.astype(np.uint64) << np.uint64(32)) | g.v.astype(np.uint64)
    claimed = np.flatnonzero(pars != M64)
    assert np.isin((pars[claimed] << np.uint64(32)) | claimed.astype(np.uint64), edges).all()   # valid in-neighbours


def test_compare_swap_test_before_swap_with_noop_swaps():
    """SHMEMG_AMO_TEST_BEFORE_SWAP when some ops have val == cond (a swap that leaves the word at cond): those ops go
    straight to the L2 atomic; per slot the result must still be a legal linearisation of CAS(cond -> val)."""
    n, slots = 1 << 18, 1 << 10
    w = World(2, slots * 8 + 4096, DEV)
    a = w.malloc(slots * 8)
    w.view(a, slots * 8, torch.int64).fill_(-1)
    key = (np.arange(n, dtype=np.int64) * 2654435761 % (2 * slots))
    val = np.arange(1, n + 1, dtype=np.uint64)
    val[::5] = M64                                                   # no-op swaps
    f = torch.empty(n, dtype=torch.int64, device=DEV)
    w.atomic_compare_swap_batch(a, to_dev((key // slots).astype(np.int32)), to_dev((key % slots).astype(np.uint32)), f,
                                cond=None, cond_scalar=M64, val=to_dev(val), flags=AMO_TEST_BEFORE_SWAP)
    w.quiet(0)
    fin = w.view(a, slots * 8, torch.int64).cpu().numpy().view(np.uint64).reshape(-1)
    fet = f.cpu().numpy().view(np.uint64)
    real = val != M64
    # ops that really swap obey the claim invariant among themselves; a no-op swap fetched cond or the final value
    check_compare_swap_claim(key[real], val[real], fet[real], fin)
    assert ((fet[~real] == M64) | (fet[~real] == fin[key[~real]])).all()


def test_c4_graph_full_scale():
    """Config 4 at its full size (RMAT scale 22, 2^26 edges, 32 PEs) in the launch configuration bench.py times."""
    g = configs.c4_graph()
    degs, pars, f_deg, f_par = _run_c4(g, AMO_HOT_AGGREGATE | AMO_TEST_BEFORE_SWAP)
    E = len(g.u)
    assert np.array_equal(degs, np.bincount(g.u, minlength=1 << 22).astype(np.uint64))   # = the oracle's pinned closed form
    ow = orc.OracleWorld(g.npes, g.verts_per_pe * 8 + 512)                           # oracle degrees, sequentially
    od = ow.malloc(g.verts_per_pe * 8)
    ow.atomic_fetch_add_batch(od, g.owner(g.u), g.local(g.u), np.ones(E, dtype=np.uint64))
    assert np.array_equal(degs, ow.view(od, g.verts_per_pe * 8, np.uint64).reshape(-1))
    check_compare_swap_claim(g.v.astype(np.int64), g.u.astype(np.uint64), f_par, pars)
    check_fetch_add(g.u.astype(np.int64), np.ones(E, dtype=np.uint64), f_deg, np.zeros(1 << 22, dtype=np.uint64), degs)


# ---- C3 ---------------------------------------------------------------------------------------------------------
def test_c3a_alltoall_full_size_and_as_put_batch():
    npes, blk = 64, 65536
    pay = configs.c3a_payload(npes, blk)
    exp = pay.reshape(npes, npes, blk).transpose(1, 0, 2).reshape(npes, npes * blk)
    w = World(npes, 3 * npes * blk + 4096, DEV)
    s, d = w.malloc(npes * blk), w.malloc(npes * blk)
    w.view(s, npes * blk).copy_(torch.from_numpy(pay))
    w.view(d, npes * blk).zero_()
    w.alltoall(d, s, blk)
    w.quiet(0)
    got = w.view(d, npes * blk).cpu().numpy()
    ow = orc.OracleWorld(npes, 2 * npes * blk + 512)
    os_, od = ow.malloc(npes * blk), ow.malloc(npes * blk)
    ow.view(os_, npes * blk)[:] = pay
    ow.alltoall(od, os_, blk)
    assert np.array_equal(got, ow.view(od, npes * blk)) and np.array_equal(got, exp)
    with pytest.raises(ShmemgError) as e:
        w.alltoall(s + blk, s, blk)
    assert e.value.code == ERR.OVERLAP
    del w
    prog = configs.c3a_put_program(npes, blk, payload=pay)       # the same exchange as 4096 puts + barrier
    w2, ld = run_gpu(prog)
    assert np.array_equal(ld.obj_numpy("dst"), exp)


@pytest.mark.parametrize("npes,blk", [(3, 1), (5, 17), (7, 4099), (16, 65536 + 48)])
def test_alltoall_ragged_sizes(npes, blk):
    w = World(npes, 2 * npes * blk + 8192, DEV)
    s = w.malloc(npes * blk + 3) + 3                             # odd base offset: byte path
    d = w.malloc(npes * blk + 5) + 5
    pay = gen.u64((npes * npes * blk + 7) // 8, 8).view(np.uint8)[:npes * npes * blk].reshape(npes, npes * blk)
    w.view(s, npes * blk).copy_(torch.from_numpy(pay))
    w.alltoall(d, s, blk)
    w.quiet(0)
    exp = pay.reshape(npes, npes, blk).transpose(1, 0, 2).reshape(npes, npes * blk)
    assert np.array_equal(w.view(d, npes * blk).cpu().numpy(), exp)


@pytest.mark.parametrize("odd", [False, True])
def test_c3b_skewed_puts(odd):
    sk = configs.c3b_skewed(odd=odd)
    w, ld = run_gpu(sk.prog)
    ow = run_oracle(sk.prog)
    assert_objects_equal(sk.prog, ld, ow)


# ---- C5 ---------------------------------------------------------------------------------------------------------
def test_c5_sum_reduce_fcollect_barrier_full_size():
    npes, nb = 128, 4 << 20
    w = World(npes, 2 * nb + 65536, DEV)
    ow = orc.OracleWorld(npes, 2 * nb + 65536)
    s, d = w.malloc(nb), w.malloc(nb)
    os_, od = ow.malloc(nb), ow.malloc(nb)
    # fp32
    x = configs.c5_f32(npes, nb // 4)
    w.view(s, nb, torch.float32).copy_(torch.from_numpy(x))
    ow.view(os_, nb, np.float32)[:] = x
    w.sum_reduce(F32, d, s, nb // 4)
    w.quiet(0)
    r64 = ow.sum_reduce_f32(od, os_, nb // 4, want_r64=True)
    g = w.view(d, nb, torch.float32).cpu().numpy()
    assert (g == g[0]).all()
    err = np.abs(g[0].astype(np.float64) - r64)
    assert (err <= 1e-6 * np.abs(r64) + 2.0 ** -36).all(), float((err / np.maximum(np.abs(r64), 1e-300)).max())
    assert np.array_equal(g, ow.view(od, nb, np.float32))        # same order, fp64 accumulate: bit-equal too
    # int64
    xi = configs.c5_i64(npes, nb // 8)
    w.view(s, nb, torch.int64).copy_(torch.from_numpy(xi))
    ow.view(os_, nb, np.int64)[:] = xi
    w.sum_reduce(I64, d, s, nb // 8)
    w.quiet(0)
    ow.sum_reduce_i64(od, os_, nb // 8)
    assert np.array_equal(w.view(d, nb, torch.int64).cpu().numpy(), ow.view(od, nb, np.int64))
    # in-place
    w.sum_reduce(I64, s, s, nb // 8)
    w.quiet(0)
    assert np.array_equal(w.view(s, nb, torch.int64).cpu().numpy()[77], ow.view(od, nb, np.int64)[0])
    # fcollect 32 KiB per PE
    fs = configs.c5_fcollect_src(npes, 32768)
    w.view(s, 32768).copy_(torch.from_numpy(fs))
    ow.view(os_, 32768)[:] = fs
    w.fcollect(d, s, 32768)
    w.quiet(0)
    ow.fcollect(od, os_, 32768)
    assert np.array_equal(w.view(d, nb).cpu().numpy(), ow.view(od, nb))
    # barriers: 10 000 stream-level barriers bump the epoch; 10 000 in-kernel barriers keep the stamp invariant
    e0 = w.barrier_epoch()
    for _ in range(200):
        w.barrier_all()
    assert w.barrier_epoch() == e0 + 200
    st = w.calloc(3, 8)
    w.barrier_all_repeat(10000, st)
    w.barrier_all_repeat(10000)
    w.quiet(0)
    sv = w.view(st, 24, torch.int64).cpu().numpy()
    assert (sv[:, 2] == 0).all(), "barrier violations: %s" % sv[:, 2]
    assert (sv[:, 0] == 10000).all() and (sv[:, 1] == 9999).all()


@pytest.mark.parametrize("npes,n,off", [(3, 1, 0), (5, 1001, 4), (9, 4097, 8), (4, 4099, 0), (2, 70000, 0), (7, 700001, 0),
                                        (33, 150001, 16)])
def test_sum_reduce_fcollect_ragged(npes, n, off):
    hb = 8 * n * (npes + 2) + 16384
    w = World(npes, hb, DEV)
    ow = orc.OracleWorld(npes, hb)
    s, d = w.malloc(8 * n + 64) + off, w.malloc(8 * npes * n + 64) + off
    os_, od = ow.malloc(8 * n + 64) + off, ow.malloc(8 * npes * n + 64) + off
    x = gen.normal_f32(npes * n, 6).reshape(npes, n)
    w.view(s, 4 * n, torch.float32).copy_(torch.from_numpy(x))
    ow.view(os_, 4 * n, np.float32)[:] = x
    w.sum_reduce(F32, d, s, n)
    ow.sum_reduce_f32(od, os_, n)
    w.quiet(0)
    assert np.array_equal(w.view(d, 4 * n, torch.float32).cpu().numpy(), ow.view(od, 4 * n, np.float32))
    if off % 8 == 0:
        xi = gen.uniform_i64(npes * n, -(1 << 40), 1 << 40, 7).reshape(npes, n)
        w.view(s, 8 * n, torch.int64).copy_(torch.from_numpy(xi))
        ow.view(os_, 8 * n, np.int64)[:] = xi
        w.sum_reduce(I64, d, s, n)
        ow.sum_reduce_i64(od, os_, n)
        w.quiet(0)
        assert np.array_equal(w.view(d, 8 * n, torch.int64).cpu().numpy(), ow.view(od, 8 * n, np.int64))
    nb = 4 * n + (1 if off == 4 else 0)                         # odd byte count exercises the byte path
    fs = gen.u64(npes * (nb // 8 + 1), 9).view(np.uint8).reshape(npes, -1)[:, :nb]
    w.view(s, nb).copy_(torch.from_numpy(np.ascontiguousarray(fs)))
    ow.view(os_, nb)[:] = fs
    w.fcollect(d, s, nb)
    ow.fcollect(od, os_, nb)
    w.quiet(0)
    assert np.array_equal(w.view(d, npes * nb).cpu().numpy(), ow.view(od, npes * nb))


# ---- C2 ---------------------------------------------------------------------------------------------------------
def _halo_run(B, rounds, consume):
    h = configs.Halo(B)
    prog = h.program(with_consume=consume)
    hb = heap_bytes_for(prog)
    w = World(8, hb, DEV)
    ld = Loaded(w, prog)
    ow = orc.OracleWorld(8, hb)
    ow.load_program(prog)
    U_off, send_off = ld.off["U"][0], ld.off["send"][0]
    ghost_off = ld.off["ghost"][0]
    fb = h.face_bytes
    sums = torch.empty(8 * 6, dtype=torch.int64, device=DEV)
    log_gpu, log_orc = [], []
    batches = [w.batch(ld.translate(h.round_ops(prog, r, consume))) for r in range(1, rounds + 1)]
    for r in range(1, rounds + 1):
        w.app_halo_perturb(U_off, B, h.seed, r)
        w.app_halo_pack(send_off, U_off, B)
        w.enqueue_batch(batches[r - 1])
        w.app_checksum64(sums, ghost_off + (r & 1) * 6 * fb, fb, 6)
        log_gpu.append(sums.cpu().numpy().view(np.uint64).copy())
        # oracle: the same round
        Uo, so = ow.obj("U", np.float64), ow.obj("send", np.float64).reshape(8, 6, B * B)
        for p in range(8):
            orc.halo_perturb(Uo[p], B, h.coord(p), h.seed, r)
            for f in range(6):
                orc.halo_pack(Uo[p], B, f, so[p, f])
        ow.run_program(h.round_ops(prog, r, consume))
        go = ow.obj("ghost", np.uint64).reshape(8, 2, 6, B * B)
        log_orc.append(np.array([orc.checksum64(go[p, r & 1, f]) for p in range(8) for f in range(6)], dtype=np.uint64))
    w.quiet(0)
    return prog, ld, ow, log_gpu, log_orc


def test_c2_halo_50_rounds_small_grid():
    prog, ld, ow, lg, lo = _halo_run(B=16, rounds=50, consume=True)
    assert_objects_equal(prog, ld, ow)                  # U, send, ghost (both parities), sig, consumed: bit-exact
    for r, (a, b) in enumerate(zip(lg, lo)):
        assert np.array_equal(a, b), "stale or wrong face in round %d" % (r + 1)


def test_c2_halo_50_rounds_b128():
    """All 50 rounds of config 2 on a 256^3 grid (128^3 blocks, 128 KiB faces): whole heap and the per-round checksum log."""
    prog, ld, ow, lg, lo = _halo_run(B=128, rounds=50, consume=False)
    assert_objects_equal(prog, ld, ow, names=["ghost", "sig", "send"])
    assert np.array_equal(ld.obj_numpy("U", np.float64), ow.obj("U", np.float64))
    assert len(lg) == 50
    for r, (a, b) in enumerate(zip(lg, lo)):
        assert np.array_equal(a, b), "stale or wrong face in round %d" % (r + 1)


def test_c2_halo_full_size_rounds():
    """Config 2 geometry at full size (512^3 grid, 256^3 blocks, 512 KiB faces), 10 rounds, whole-heap oracle compare and
    the checksum log of every round."""
    prog, ld, ow, lg, lo = _halo_run(B=256, rounds=10, consume=False)
    assert_objects_equal(prog, ld, ow, names=["ghost", "sig", "send"])
    assert np.array_equal(ld.obj_numpy("U", np.float64), ow.obj("U", np.float64))
    for a, b in zip(lg, lo):
        assert np.array_equal(a, b)


def test_c1_final_array_matches_the_stored_oracle_checksum():
    """tests/golden/oracle_checksums.txt is written from the oracle alone; the CUDA path must land on the same bytes."""
    import hashlib
    import os
    stored = dict(ln.split() for ln in open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden",
                                                         "oracle_checksums.txt")) if ln.strip() and ln[0] != "#")
    wl = configs.c1_atomic_add()
    w = World(wl.npes, wl.nelem * 8 + 4096, DEV)
    a = w.calloc(wl.nelem, 8)
    w.atomic_add_batch(a, to_dev(wl.tgt_pe), to_dev(wl.idx.astype(np.int64)), val=to_dev(wl.val))
    w.quiet(0); w.barrier_all()
    got = hashlib.sha256(w.view(a, wl.nelem * 8).cpu().numpy().tobytes()).hexdigest()[:32]
    assert got == stored["c1_atomic_add_full"]
