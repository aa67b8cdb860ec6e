"""GPU parity of the ONE-CALL batch form (shmemg_enqueue_batch: device-resident descriptors planned on the device; SURVEY.md
8(a) a5 / 8(b)): every program the host-planned batches run is run through it and compared with the
CPU oracle; the device planner's records are compared WORD FOR WORD with the host planner's; status reporting; descriptors
generated on the GPU."""
import numpy as np
import pytest
import torch

from gpu_common import DEV, assert_objects_equal, heap_bytes_for, ops_to_dev, run_gpu, run_gpu_onecall, run_oracle
from invariants import check_compare_swap_claim, check_fetch_add
from litmus_model import enumerate_outcomes, to_spec_program
from paper_2607_08006_b200 import CMP, ERR, OP, OP_DTYPE, ShmemgError, World
from paper_2607_08006_b200.loader import Loaded
from test_gpu_batch import TINY
from workloads import configs, gen, litmus
from workloads.spec import Program

pytestmark = pytest.mark.gpu
M64 = (1 << 64) - 1

LITMUS = {
    "mp_fence": lambda: litmus.mp_fence(),
    "mp_fence_big": lambda: litmus.mp_fence(npes=64, rounds=6, nbytes=300000, lag=1),
    "mp_quiet3": lambda: litmus.mp_quiet_third_party(),
    "put_signal_sizes": lambda: litmus.put_signal_sizes(),
    "signal_add_fanin": lambda: litmus.signal_add_fanin(),
    "barrier_stamp": lambda: litmus.barrier_stamp(),
    "barrier_stamp128": lambda: litmus.barrier_stamp(npes=128, rounds=12),
    "wait_after_wait": lambda: litmus.wait_after_wait(),
    "two_contexts": lambda: litmus.two_contexts(),
    "contexts_amos_waits": lambda: litmus.contexts_amos_waits(),
}


@pytest.mark.parametrize("name", sorted(LITMUS))
def test_litmus_programs_one_call_match_oracle(name):
    prog = LITMUS[name]()
    w, ld = run_gpu_onecall(prog)
    assert_objects_equal(prog, ld, run_oracle(prog))


def random_put_get(npes=6, nops=400, slot=5000, seed=3):
    rng = np.random.default_rng(seed)
    prog = Program(npes)
    prog.obj("src", 40000, gen.u64(npes * 40000 // 8, 77).view(np.uint8).reshape(npes, 40000))
    prog.obj("dst", nops * slot)
    for k in range(nops):
        i, t = int(rng.integers(npes)), int(rng.integers(npes))
        n = int(rng.integers(0, slot - 32))
        s, d = int(rng.integers(0, 40000 - n)), k * slot + int(rng.integers(0, 32))
        if k % 4 == 1:
            s = (s & ~15) + (d & 15)                               # congruent mod 16: head + bulk body + tail
        (prog.put if k % 2 else prog.get)(i, t, ("dst", d), ("src", s), n)
    return prog


def test_random_put_get_unaligned_one_call():
    prog = random_put_get()
    w, ld = run_gpu_onecall(prog)
    assert_objects_equal(prog, ld, run_oracle(prog))


def test_random_amos_one_call():
    prog = litmus.random_amos()
    w, ld = run_gpu_onecall(prog)
    ow = run_oracle(prog)
    ops = prog.ops
    nw = prog.obj_bytes[0] // 8
    words = ld.obj_numpy("words", np.uint64)
    assert np.array_equal(words[:, :nw // 2], ow.obj("words", np.uint64)[:, :nw // 2])
    assert np.array_equal(words[:, nw // 2:] == M64, ow.obj("words", np.uint64)[:, nw // 2:] == M64)
    fetch = ld.obj_numpy("fetch", np.uint64)
    key = ops["target"].astype(np.int64) * nw + (ops["rem_off"] // 8).astype(np.int64)
    fa, ad, cs = ops["kind"] == 5, ops["kind"] == 4, ops["kind"] == 6
    fetched = fetch[ops["initiator"], np.arange(len(ops))]
    sel = fa & ~np.isin(key, np.unique(key[ad]))
    init = np.zeros(prog.npes * nw, dtype=np.uint64)
    init.reshape(prog.npes, nw)[:, nw // 2:] = M64
    fin = words.reshape(-1)
    sub_final = init.copy()
    ks = np.unique(key[sel])
    sub_final[ks] = fin[ks]
    check_fetch_add(key[sel], ops["value"][sel], fetched[sel], init, sub_final)
    cas_final = np.full(prog.npes * nw, M64, dtype=np.uint64)
    kc = np.unique(key[cs])
    cas_final[kc] = fin[kc]
    check_compare_swap_claim(key[cs], ops["value"][cs], fetched[cs], cas_final)


@pytest.mark.parametrize("name", sorted(TINY))
def test_tiny_programs_one_call_land_in_enumerated_outcome_set(name):
    prog, init, order = TINY[name]
    allowed = enumerate_outcomes(prog, init)
    sp = to_spec_program(prog, init, order)
    for k in range(4):
        w, ld = run_gpu_onecall(sp, arena=bool(k & 1))
        got = tuple(tuple(int(x) for x in row) for row in ld.obj_numpy("w", np.uint64))
        assert got in allowed, (name, got)


# ---- the device planner writes the host planner's plan, word for word -------------------------------------------------------
def plans(w, ops):
    """(tile records, AMO / wait records) of the host plan and of the device plan, tile.src of AMO / wait runs made relative."""
    b = w.batch(ops)
    hp = b.plan.cpu().numpy()
    payload = int(ops["nbytes"][(ops["opcode"] >= 1) & (ops["opcode"] <= 3)].sum())
    work = torch.empty(w.batch_work_bytes(len(ops), payload), dtype=torch.uint8, device=DEV)
    # plan only: a program of the tests would also run, which is harmless, but the wait of an unsatisfied program would hang
    w.enqueue_batch_dev(ops_to_dev(ops), len(ops), work)
    assert w.batch_status(work) == (0, 0)
    w.quiet(0)
    dp = work.cpu().numpy()

    def parse(raw, base_addr):
        ntiles, nunits = (int(x) for x in raw[:8].view(np.uint32))
        all_total = int(raw[24:28].view(np.uint32)[0])
        tiles_off, aux_off = (int(x) for x in raw[32:48].view(np.uint64))
        tiles = raw[tiles_off:tiles_off + 64 * ntiles].reshape(ntiles, 64).copy()
        kind = tiles[:, 36:40].copy().view(np.uint32).reshape(-1) & 0xff
        runs = (kind == 3) | (kind == 4)
        naux = int(tiles[runs, 32:36].copy().view(np.uint32).sum())
        src = tiles[:, 8:16].copy().view(np.uint64).reshape(-1)
        src[runs] = (src[runs] - np.uint64(base_addr + aux_off)) // np.uint64(64)
        tiles[:, 8:16] = src.view(np.uint8).reshape(-1, 8)
        aux = raw[aux_off:aux_off + 64 * naux].reshape(naux, 64).copy()
        # pe_total (how far done[domain] advances per launch) only serves the re-launch of a host plan: a one-call plan
        # starts its counters at zero in every call and leaves the field 0
        tiles[:, 60:64] = 0
        aux[:, 48:52] = 0
        return ntiles, nunits, all_total, tiles, aux
    return parse(hp, b.plan.data_ptr()), parse(dp, work.data_ptr()), (int(dp[80:84].view(np.uint32)[0]), int(dp[84:88].view(np.uint32)[0]))


def host_ring(ops, sm=148):
    bulk = int(ops["nbytes"][(ops["opcode"] >= 1) & (ops["opcode"] <= 3)].sum())
    return (16384, 12) if bulk <= 256 * 1024 * sm else (32768, 7)


PLAN_CASES = dict(LITMUS)
PLAN_CASES.update({
    "random_put_get": random_put_get,
    "random_amos": lambda: litmus.random_amos(n_ops=3000),
    "c3a_puts": lambda: configs.c3a_put_program(16, 65536),
    "c3b_zipf": lambda: configs.c3b_skewed().prog,
    "c3b_zipf_odd": lambda: configs.c3b_skewed(npes=16, odd=True).prog,
})


@pytest.mark.parametrize("name", sorted(PLAN_CASES))
def test_device_plan_equals_host_plan(name):
    prog = PLAN_CASES[name]()
    w = World(prog.npes, heap_bytes_for(prog), DEV)
    ld = Loaded(w, prog)
    ops = ld.translate(prog)
    (hn, hu, ha, ht, hx), (dn, du, da, dt, dx), ring = plans(w, ops)
    assert (hn, hu, ha) == (dn, du, da), "ntiles / nunits / all_total"
    assert np.array_equal(ht, dt), "tile records differ first at %s" % (np.argwhere(ht != dt)[:1],)
    assert np.array_equal(hx, dx), "AMO / wait records differ first at %s" % (np.argwhere(hx != dx)[:1],)
    assert ring == host_ring(ops)


def test_device_plan_equals_host_plan_halo_rounds():
    h = configs.Halo(64)
    prog = h.program(with_consume=True, with_U=False)
    w = World(8, heap_bytes_for(prog), DEV)
    ld = Loaded(w, prog)
    ld.obj("sig").fill_(255)                                         # every wait (GE round) is satisfied at once
    for r in (1, 2):
        ops = ld.translate(h.round_ops(prog, r, True))
        (hn, hu, ha, ht, hx), (dn, du, da, dt, dx), ring = plans(w, ops)
        assert (hn, hu, ha) == (dn, du, da) and np.array_equal(ht, dt) and np.array_equal(hx, dx)


# ---- status reporting, workspace reuse, descriptors generated on the GPU ------------------------------------------------------
def test_bad_descriptor_and_small_workspace_are_reported_and_nothing_runs():
    w = World(2, 20 << 20, DEV)
    a = w.malloc(18 << 20)
    w.view(a, 18 << 20).zero_()
    w.view(a, 4096)[0].fill_(7)
    ops = np.zeros(3, dtype=OP_DTYPE)
    ops["opcode"] = OP.PUT
    ops["target_pe"] = [1, 1, 2]                                      # op 2: target PE out of range
    ops["rem_off"] = [a + 4096, a + 8192, a]
    ops["loc_off"] = a
    ops["nbytes"] = 4096
    w.enqueue_batch_dev(ops_to_dev(ops), 3)
    assert w.batch_status() == (ERR.PE, 2)
    assert int(w.view(a, 1 << 19)[1].sum()) == 0                      # the two valid puts did not run either
    ops["target_pe"][2] = 1
    ops["opcode"][1] = OP.ATOMIC_ADD
    ops["rem_off"][1] = a + 12                                        # misaligned AMO word: the FIRST bad op is reported
    ops["opcode"][2] = 77
    w.enqueue_batch_dev(ops_to_dev(ops), 3)
    assert w.batch_status() == (ERR.ALIGN, 1)
    # a workspace that holds the per-op records but not the 512 tile records of an 8 MiB relatively misaligned put
    n = 8 << 20
    ops = np.zeros(1, dtype=OP_DTYPE)
    ops["opcode"], ops["target_pe"], ops["rem_off"], ops["loc_off"], ops["nbytes"] = OP.PUT, 1, a + (9 << 20) + 1, a, n
    small = torch.empty(w.batch_work_bytes(1, 0), dtype=torch.uint8, device=DEV)
    w.enqueue_batch_dev(ops_to_dev(ops), 1, small)
    st, need = w.batch_status(small)
    assert st == ERR.NOMEM and need == n // 16384
    assert int(w.view(a, 18 << 20)[1].sum()) == 0
    big = torch.empty(w.batch_work_bytes(1, n), dtype=torch.uint8, device=DEV)
    w.enqueue_batch_dev(ops_to_dev(ops), 1, big)
    assert w.batch_status(big) == (0, 0)
    assert int(w.view(a, 18 << 20)[1].sum()) == 7 * 4096
    # host-checkable misuse
    with pytest.raises(ShmemgError):
        w.enqueue_batch_dev(ops_to_dev(ops), 1, torch.empty(512, dtype=torch.uint8, device=DEV))
    w.enqueue_batch_dev(torch.zeros(64, dtype=torch.uint8, device=DEV), 0)      # empty batch: nothing enqueued


def test_workspace_is_reused_and_stream_order_holds():
    """Batch B after batch A on one stream, same workspace: B is planned after A has finished and reads what A wrote."""
    npes, blk = 8, 20000
    a = configs.c3a_put_program(npes, blk)
    b = a.fork()
    for i in range(npes):
        for j in range(npes):
            b.put(i, j, ("src", i * blk), ("dst", j * blk), blk)
    w = World(npes, heap_bytes_for(a), DEV)
    ld = Loaded(w, a)
    oa, ob = ops_to_dev(ld.translate(a)), ops_to_dev(ld.translate(b))
    src0 = ld.obj_numpy("src").copy()
    for _ in range(3):
        w.enqueue_batch_dev(oa, len(a))
        w.enqueue_batch_dev(ob, len(b))
    assert w.batch_status() == (0, 0)
    exp_dst = src0.reshape(npes, npes, blk).transpose(1, 0, 2).reshape(npes, npes * blk)
    assert np.array_equal(ld.obj_numpy("dst"), exp_dst)
    assert np.array_equal(ld.obj_numpy("src"), src0)


def test_descriptors_generated_on_the_gpu():
    """The op list is produced by device code (torch kernels on the same stream) and never exists on the host: a ring shift
    of `cnt[p]` bytes per PE where cnt is itself device data (fine-grained updates generated by GPU kernels)."""
    npes, cap = 16, 1 << 16
    w = World(npes, 4 * cap, DEV)
    src, dst = w.malloc(cap), w.malloc(cap)
    pay = gen.u64(npes * cap // 8, 5).view(np.uint8).reshape(npes, cap)
    w.view(src, cap).copy_(torch.from_numpy(pay))
    w.view(dst, cap).zero_()
    cnt = (torch.arange(npes, device=DEV, dtype=torch.int64) * 3797 + 123) % cap          # device-resident sizes
    rec = torch.zeros(npes, 8, dtype=torch.int64, device=DEV)                              # 64-byte records as 8 x int64
    pe = torch.arange(npes, device=DEV, dtype=torch.int64)
    rec[:, 0] = OP.PUT | (pe << 32)                                                       # opcode | initiator_pe << 32
    rec[:, 1] = (pe + 1) % npes                                                            # target_pe
    rec[:, 2], rec[:, 3], rec[:, 4] = dst, src, cnt
    w.enqueue_batch_dev(rec.view(torch.uint8).reshape(-1), npes)
    assert w.batch_status() == (0, 0)
    got, c = w.view(dst, cap).cpu().numpy(), cnt.cpu().numpy()
    for p in range(npes):
        t = (p + 1) % npes
        assert np.array_equal(got[t, :c[p]], pay[p, :c[p]]) and not got[t, c[p]:].any()


def test_onecall_batches_captured_in_a_cuda_graph():
    """shmemg_enqueue_batch is two kernel launches and nothing else (no host pass, no synchronisation, no allocation), so a
    sequence of one-call batches can be captured in a CUDA graph; every replay plans the descriptors again on the device (the
    descriptor array is re-read: it is changed between the replays here) and the batches stay stream-ordered inside the graph."""
    npes, blk = 8, 20000
    a = configs.c3a_put_program(npes, blk)                       # src -> dst (transpose)
    b = a.fork()
    for i in range(npes):
        for j in range(npes):
            b.put(i, j, ("src", i * blk), ("dst", j * blk), blk)   # dst -> src (transpose back)
    while len(b.ops) < len(a.ops):
        b.barrier_all()                                          # same number of descriptors as `a` (which ends with a barrier)
    w = World(npes, heap_bytes_for(a), DEV)
    ld = Loaded(w, a)
    oa, ob = ld.translate(a), ld.translate(b)
    assert len(oa) == len(ob)
    da, db = ops_to_dev(oa), ops_to_dev(ob)
    work = torch.empty(w.batch_work_bytes(len(oa), int(oa["nbytes"].sum())), dtype=torch.uint8, device=DEV)
    src0 = ld.obj_numpy("src").copy()
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        w.enqueue_batch_dev(da, len(oa), work)                   # warm-up outside the capture (function attributes)
        w.enqueue_batch_dev(db, len(ob), work)
        torch.cuda.synchronize()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=s):
            for _ in range(3):
                w.enqueue_batch_dev(da, len(oa), work)
                w.enqueue_batch_dev(db, len(ob), work)
            w.enqueue_batch_dev(da, len(oa), work)
        g.replay()
        torch.cuda.synchronize()
        assert w.batch_status(work) == (0, 0)
        exp_dst = src0.reshape(npes, npes, blk).transpose(1, 0, 2).reshape(npes, npes * blk)
        assert np.array_equal(ld.obj_numpy("dst"), exp_dst) and np.array_equal(ld.obj_numpy("src"), src0)
        # the descriptors are device data read at replay time: make the LAST batch of the graph the back-transpose too
        ld.obj("dst").copy_(torch.from_numpy(exp_dst))
        ld.obj("src").zero_()
        da.copy_(db)
        g.replay()
        torch.cuda.synchronize()
    assert np.array_equal(ld.obj_numpy("src"), src0)              # every batch of this replay was dst -> src


@pytest.mark.parametrize("form", ["pre-planned", "one-call"])
def test_signal_produced_by_one_batch_and_awaited_by_the_next(form):
    """Every executor launch starts as a programmatic dependent of the kernel before it: its CTAs may be resident while the
    previous batch still runs.  A batch that WAITS for a signal the previous batch sets, and then forwards the payload, must
    still see signal and payload (nothing mutable is touched before griddepcontrol.wait).  20 rounds back to back."""
    npes, n = 6, 30000
    prog = Program(npes)
    prog.obj("src", n, gen.u64(npes * n // 8, 17).view(np.uint8).reshape(npes, n))
    prog.obj("mid", n)
    prog.obj("dst", n)
    prog.obj("sig", 8)
    batches = []
    for r in range(1, 21):
        b1 = prog.fork()
        for i in range(npes):
            b1.put_signal(i, (i + 1) % npes, ("mid", 0), ("src", 0), n - r, ("sig", 0), r)
        b2 = prog.fork()
        for i in range(npes):
            b2.signal_wait_until(i, ("sig", 0), CMP.GE, r)
            b2.put(i, (i + 2) % npes, ("dst", 0), ("mid", 0), n - r)
        batches += [b1, b2]
    w, ld = (run_gpu if form == "pre-planned" else run_gpu_onecall)(prog, batches=batches)
    ow = run_oracle(prog, batches=batches)
    assert_objects_equal(prog, ld, ow)
