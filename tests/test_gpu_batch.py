"""GPU parity: the batch executor (put/get/put_signal/wait/fence/quiet/barrier/AMOs through descriptors)
against the CPU oracle, element by element, plus the brute-force outcome sets for tiny programs."""
import numpy as np
import pytest
import torch

from gpu_common import DEV, assert_objects_equal, heap_bytes_for, ops_to_dev, run_gpu, run_oracle
from invariants import check_compare_swap_claim, check_fetch_add
from litmus_model import enumerate_outcomes, to_spec_program
from paper_2607_08006_b200 import CMP, ERR, OP, OP_DTYPE, ShmemgError, World
from paper_2607_08006_b200.loader import Loaded
from workloads import configs, gen, litmus
from workloads.spec import SIGNAL_ADD, Program

pytestmark = pytest.mark.gpu
M64 = (1 << 64) - 1


@pytest.mark.parametrize("make", [
    lambda: litmus.mp_fence(),
    lambda: litmus.mp_fence(npes=64, rounds=6, nbytes=300000, lag=1),
    lambda: litmus.mp_quiet_third_party(),
    lambda: litmus.put_signal_sizes(),
    lambda: litmus.signal_add_fanin(),
    lambda: litmus.barrier_stamp(),
    lambda: litmus.barrier_stamp(npes=128, rounds=12),
    lambda: litmus.wait_after_wait(),
    lambda: litmus.two_contexts(),
    lambda: litmus.contexts_amos_waits(),
], ids=["mp_fence", "mp_fence_big", "mp_quiet3", "put_signal_sizes", "signal_add_fanin", "barrier_stamp",
        "barrier_stamp128", "wait_after_wait", "two_contexts", "contexts_amos_waits"])
def test_litmus_programs_match_oracle(make):
    prog = make()
    w, ld = run_gpu(prog)
    ow = run_oracle(prog)
    assert_objects_equal(prog, ld, ow)


def test_barrier_stamp_log_is_round_numbers():
    prog = litmus.barrier_stamp(npes=16, rounds=30)
    w, ld = run_gpu(prog)
    log = ld.obj_numpy("log", np.uint64)
    assert (log[:, 1:] == np.arange(1, 31, dtype=np.uint64)).all()


def test_random_put_get_program_unaligned():
    """Race-free random puts/gets with arbitrary sizes and alignments: each op owns a private dest slot."""
    npes, nops, slot = 6, 400, 5000
    rng = np.random.default_rng(3)
    prog = Program(npes)
    src = gen.u64(npes * 40000 // 8, 77).view(np.uint8).reshape(npes, 40000)
    prog.obj("src", 40000, src)
    prog.obj("dst", nops * slot)
    for k in range(nops):
        i, t = int(rng.integers(npes)), int(rng.integers(npes))
        n = int(rng.integers(0, slot - 32))
        s, d = int(rng.integers(0, 40000 - n)), k * slot + int(rng.integers(0, 32))
        if k % 2:
            prog.put(i, t, ("dst", d), ("src", s), n)
        else:
            prog.get(i, t, ("dst", d), ("src", s), n)
    w, ld = run_gpu(prog)
    assert_objects_equal(prog, ld, run_oracle(prog))


def test_random_amos_through_descriptors():
    prog = litmus.random_amos()
    w, ld = run_gpu(prog)
    ow = run_oracle(prog)
    ops = prog.ops
    nw = prog.obj_bytes[0] // 8
    words = ld.obj_numpy("words", np.uint64)
    # add / fetch-add finals are schedule independent: bit-exact vs the oracle; CAS winners are not (invariants below)
    assert np.array_equal(words[:, :nw // 2], ow.obj("words", np.uint64)[:, :nw // 2])
    assert np.array_equal(words[:, nw // 2:] == M64, ow.obj("words", np.uint64)[:, nw // 2:] == M64)
    fetch = ld.obj_numpy("fetch", np.uint64)
    key = ops["target"].astype(np.int64) * nw + (ops["rem_off"] // 8).astype(np.int64)
    fa = ops["kind"] == 5
    ad = ops["kind"] == 4
    cs = ops["kind"] == 6
    idx = np.arange(len(ops))
    fetched = fetch[ops["initiator"], idx]                        # op i's private slot in its initiator's heap
    # fetch-add invariant needs every update of the word: treat plain adds as unobserved updates by checking
    # only words that received no plain add
    plain_words = np.unique(key[ad])
    sel = fa & ~np.isin(key, plain_words)
    init = np.zeros(prog.npes * nw, dtype=np.uint64)
    init.reshape(prog.npes, nw)[:, nw // 2:] = M64
    fin = words.reshape(-1)
    if sel.any():
        sub_final = init.copy()
        ks = np.unique(key[sel])
        sub_final[ks] = fin[ks]
        check_fetch_add(key[sel], ops["value"][sel], fetched[sel], init, sub_final)
    cas_final = np.full(prog.npes * nw, M64, dtype=np.uint64)
    kc = np.unique(key[cs])
    cas_final[kc] = fin[kc]
    check_compare_swap_claim(key[cs], ops["value"][cs], fetched[cs], cas_final)


TINY = {
    "mp_fence": ([[("put", 1, 0, 2), ("fence",), ("put", 1, 1, 3)], [("wait", 1, "eq", 1), ("get", 1, 4, 0)]],
                 [[0, 0, 42, 1, 0], [0] * 5], [0, 0, 0, 1, 1]),
    "mp_no_fence": ([[("put", 1, 0, 2), ("put", 1, 1, 3)], [("wait", 1, "eq", 1), ("get", 1, 4, 0)]],
                    [[0, 0, 42, 1, 0], [0] * 5], [0, 0, 1, 1]),
    "quiet_third_party": ([[("put", 1, 0, 2), ("quiet",), ("put", 2, 1, 3)], [],
                           [("wait", 1, "eq", 1), ("get", 1, 4, 0)]],
                          [[0, 0, 42, 1, 0], [0] * 5, [0] * 5], [0, 0, 0, 2, 2]),
    "put_signal": ([[("put_signal", 1, 0, 2, 1, 9, "set")], [("wait", 1, "eq", 9), ("get", 1, 4, 0)]],
                   [[0, 0, 42, 1, 0], [0] * 5], [0, 1, 1]),
    "fadd_fadd": ([[("fadd", 1, 0, 2, 1)], [("fadd", 1, 0, 3, 1)]], [[0, 0], [0, 0]], [0, 1]),
    "cas_cas": ([[("cas", 1, 0, M64, 100, 1)], [("cas", 1, 0, M64, 200, 1)]], [[M64, 0], [M64, 0]], [0, 1]),
    "barrier": ([[("put", 1, 0, 2), ("barrier",), ("get", 0, 4, 0)], [("put", 0, 0, 2), ("barrier",), ("get", 1, 4, 0)]],
                [[0, 0, 42, 0, 0], [0, 0, 43, 0, 0]], [0, 1, 0, 1, 0, 1]),
    "quiet_readback": ([[("put", 1, 0, 2), ("quiet",), ("get", 1, 4, 0)], []], [[0, 0, 42, 0, 0], [0] * 5], [0, 0, 0]),
    # contexts (ctx > 0) with waits and fetching AMOs: fetch slots and wait words live in the PE's window, not the domain's
    "ctx_quiet_independent": ([[("put", 1, 0, 2, "@0"), ("put", 1, 5, 5, "@1"), ("quiet", "@1"), ("put", 1, 1, 3, "@1")],
                               [("wait", 1, "eq", 1, "@2"), ("get", 1, 4, 0, "@2")]],
                              [[0, 0, 42, 1, 0, 7], [0] * 6], [0, 0, 0, 0, 1, 1]),
    "ctx_fadd_cas_wait": ([[("fadd", 1, 0, 2, 1, "@3"), ("cas", 1, 2, M64, 9, 3, "@3"), ("quiet", "@3"), ("add", 1, 4, 1, "@3")],
                           [("wait", 4, "ge", 1, "@1"), ("fadd", 1, 0, 5, 1, "@1"), ("cas", 1, 2, M64, 8, 3, "@1")]],
                          [[0, 0, 0, 0, 0], [0, 0, M64, 0, 0]], [0, 0, 0, 0, 1, 1, 1]),
    # a wait on context 0 followed by a put of the received word on context 1 (shmemg.h "Batch semantics": in a batch the wait
    # orders only its own context, so the forward may carry the old word; the device-initiated interpreter blocks the whole PE)
    "ctx_wait_then_forward_on_other_ctx": ([[("put", 1, 0, 2), ("fence",), ("put", 1, 1, 3)],
                                            [("wait", 1, "eq", 1, "@0"), ("put", 0, 4, 0, "@1")]],
                                           [[0, 0, 42, 1, 0], [0] * 5], [0, 0, 0, 1, 1]),
    # ... and the portable form: a wait on the forwarding context too
    "ctx_wait_on_both_then_forward": ([[("put", 1, 0, 2), ("fence",), ("put", 1, 1, 3)],
                                       [("wait", 1, "eq", 1, "@0"), ("wait", 1, "eq", 1, "@1"), ("put", 0, 4, 0, "@1")]],
                                      [[0, 0, 42, 1, 0], [0] * 5], [0, 0, 0, 1, 1, 1]),
    "add_fence_add": ([[("add", 1, 0, 7), ("fence",), ("add", 1, 1, 1)], [("wait", 1, "ge", 1), ("get", 1, 4, 0)]],
                      [[0] * 5, [0] * 5], [0, 0, 0, 1, 1]),
}


@pytest.mark.parametrize("name", sorted(TINY))
def test_tiny_programs_land_in_enumerated_outcome_set(name):
    """The GPU's final state must be one of the states the ordering rules allow (brute force)."""
    prog, init, order = TINY[name]
    allowed = enumerate_outcomes(prog, init)
    sp = to_spec_program(prog, init, order)
    for _ in range(5):
        w, ld = run_gpu(sp)
        got = tuple(tuple(int(x) for x in row) for row in ld.obj_numpy("w", np.uint64))
        assert got in allowed, (name, got)


@pytest.mark.parametrize("onecall", [False, True])
def test_dependent_launch_can_be_turned_off(onecall):
    """shmemg_set_dependent_launch(w, 0): plain stream-ordered launches of the executor (and of the device planner in the
    one-call form).  Same results: a program whose second batch awaits signals raised by the first, back to back on one stream."""
    prog = litmus.wait_after_wait(npes=4, groups=3, chain=8, nbytes=1 << 16)
    ow = run_oracle(prog)
    w = World(prog.npes, heap_bytes_for(prog), DEV)
    w.set_dependent_launch(False)
    ld = Loaded(w, prog)
    ops = ld.translate(prog)
    half = len(ops) // 2
    keep = []
    for part in (ops[:half], ops[half:]):
        if onecall:
            od = ops_to_dev(part)
            w.enqueue_batch_dev(od, len(part), None)
            keep.append(od)
        else:
            keep.append(w.batch(part))
            w.enqueue_batch(keep[-1])
    w.quiet(0)
    assert_objects_equal(prog, ld, ow)
    w.set_dependent_launch(True)


def test_batch_can_be_enqueued_repeatedly_and_stream_order_holds():
    """Stream ordering: batch B enqueued after batch A on one stream reads everything A wrote;
    an idempotent batch can be replayed (the last CTA re-arms the plan)."""
    npes, blk = 8, 20000
    a = configs.c3a_put_program(npes, blk)                       # src -> dst (transpose)
    b = a.fork()
    b.obj_names = a.obj_names
    for i in range(npes):
        for j in range(npes):
            b.put(i, j, ("src", i * blk), ("dst", j * blk), blk)   # dst -> src (transpose back)
    hb = heap_bytes_for(a)
    w = World(npes, hb, DEV)
    ld = Loaded(w, a)
    ba, bb = w.batch(ld.translate(a)), w.batch(ld.translate(b))
    src0 = ld.obj_numpy("src").copy()
    for _ in range(3):
        w.enqueue_batch(ba)
        w.enqueue_batch(bb)
    w.quiet(0)
    exp_dst = src0.reshape(npes, npes, blk).transpose(1, 0, 2).reshape(npes, npes * blk)
    assert np.array_equal(ld.obj_numpy("dst"), exp_dst)
    assert np.array_equal(ld.obj_numpy("src"), src0)              # transpose of transpose


def test_batches_captured_in_a_cuda_graph_replay_with_stream_order():
    """A pre-planned batch is re-enqueueable (monotonic counters), so its launch can be captured in a CUDA graph and replayed.
    Every executor launch is a programmatic dependent of the kernel before it (griddepcontrol.wait before anything mutable is
    touched): inside the graph, batch B must still read everything batch A wrote, replay after replay."""
    npes, blk = 8, 20000
    a = configs.c3a_put_program(npes, blk)                       # src -> dst (transpose)
    a.obj("sig", 8 * npes)
    b = a.fork()
    for i in range(npes):
        for j in range(npes):
            b.put_signal(i, j, ("src", i * blk), ("dst", j * blk), blk, ("sig", 8 * i), 1, SIGNAL_ADD)   # dst -> src, counted
    w = World(npes, heap_bytes_for(a), DEV)
    ld = Loaded(w, a)
    ba, bb = w.batch(ld.translate(a)), w.batch(ld.translate(b))
    src0 = ld.obj_numpy("src").copy()
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        w.enqueue_batch(ba)                                      # warm-up outside the capture (module load, attributes)
        w.enqueue_batch(bb)
        torch.cuda.synchronize()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=s):
            for _ in range(5):
                w.enqueue_batch(ba)
                w.enqueue_batch(bb)
        for _ in range(3):
            g.replay()
        w.quiet(0)
    torch.cuda.synchronize()
    exp_dst = src0.reshape(npes, npes, blk).transpose(1, 0, 2).reshape(npes, npes * blk)
    assert np.array_equal(ld.obj_numpy("dst"), exp_dst)
    assert np.array_equal(ld.obj_numpy("src"), src0)              # transpose of transpose, 16 times over
    assert (ld.obj_numpy("sig", np.uint64) == 16).all()           # every put_signal of each of the 16 launches signalled once


def test_edge_cases_empty_and_zero_byte():
    w = World(4, 1 << 16, DEV)
    b = w.batch(np.zeros(0, dtype=OP_DTYPE))
    w.enqueue_batch(b)
    a = w.calloc(64, 8)
    ops = np.zeros(3, dtype=OP_DTYPE)
    ops["opcode"] = [OP.PUT, OP.PUT_SIGNAL, OP.SIGNAL_WAIT_UNTIL]
    ops["initiator_pe"] = [0, 0, 1]
    ops["target_pe"] = [1, 1, 1]
    ops["rem_off"] = a
    ops["loc_off"] = [a, a, a + 8]
    ops["nbytes"] = 0                                             # zero-byte put and zero-byte put_signal
    ops["sig_off"] = a + 8
    ops["value"] = [0, 5, 5]
    ops["cmp"] = CMP.EQ
    w.enqueue_batch(w.batch(ops))
    w.quiet(0)
    v = w.view(a, 64 * 8, torch.int64).cpu().numpy()
    assert v[1, 1] == 5 and v.sum() == 5
    only_markers = np.zeros(3, dtype=OP_DTYPE)
    only_markers["opcode"] = [OP.FENCE, OP.QUIET, OP.BARRIER_ALL]
    w.enqueue_batch(w.batch(only_markers))
    w.quiet(0)


def test_bad_descriptors_are_rejected_on_the_host():
    w = World(2, 4096, DEV)
    def one(**kw):
        o = np.zeros(1, dtype=OP_DTYPE)
        for k, v in kw.items():
            o[k] = v
        return o
    for kw, code in [
        (dict(opcode=OP.PUT, target_pe=2, nbytes=8), ERR.PE),
        (dict(opcode=OP.PUT, target_pe=1, rem_off=4090, nbytes=8), ERR.RANGE),
        (dict(opcode=OP.ATOMIC_ADD, target_pe=1, rem_off=12), ERR.ALIGN),
        (dict(opcode=OP.PUT_SIGNAL, target_pe=1, nbytes=8, sig_off=4), ERR.ALIGN),
        (dict(opcode=OP.SIGNAL_WAIT_UNTIL, cmp=9), ERR.ARG),
        (dict(opcode=77), ERR.ARG),
        (dict(opcode=OP.FENCE, initiator_pe=5), ERR.PE),
    ]:
        with pytest.raises(ShmemgError) as e:
            w.batch(one(**kw))
        assert e.value.code == code, (kw, e.value)


def test_context_field_is_validated_and_quiet_is_per_context():
    """ctx >= SHMEMG_CTX_MAX is rejected; a QUIET on an unused context orders nothing but is legal."""
    from workloads.spec import SIGNAL_ADD, Program
    w = World(2, 1 << 16, DEV)
    a = w.malloc(4096)
    ops = np.zeros(3, dtype=OP_DTYPE)
    ops["opcode"] = [OP.PUT, OP.QUIET, OP.PUT]
    ops["initiator_pe"] = [0, 0, 0]
    ops["target_pe"] = [1, 0, 1]
    ops["rem_off"] = [a, 0, a + 64]
    ops["loc_off"] = [a + 128, 0, a + 256]
    ops["nbytes"] = [64, 0, 64]
    ops["ctx"] = [0, 7, 3]
    w.view(a, 4096).copy_(torch.arange(4096, device=DEV).to(torch.uint8).repeat(2, 1))
    b = w.batch(ops)
    w.enqueue_batch(b)
    w.quiet(0)
    v = w.view(a, 4096).cpu().numpy()
    assert np.array_equal(v[1, :64], v[0, 128:192]) and np.array_equal(v[1, 64:128], v[0, 256:320])
    ops["ctx"][1] = 8
    with pytest.raises(ShmemgError):
        w.batch(ops)


def test_quiet_on_one_context_does_not_depend_on_the_other():
    """White-box check of the plan (tile records, 64 B each after the 256-byte header; dependency threshold at byte 52,
    ordering domain at byte 48): the flag put behind QUIET(ctx 1) waits for ONE op (the small put of ctx 1) in domain
    npes + pe, not for the four bulk puts of ctx 0; with everything on ctx 0 it waits for all five."""
    w = World(4, 8 << 20, DEV)
    a = w.malloc(6 << 20)

    def plan(ctx_small):
        ops = np.zeros(7, dtype=OP_DTYPE)
        ops["opcode"] = [OP.PUT] * 4 + [OP.PUT, OP.QUIET, OP.PUT]
        ops["initiator_pe"] = 2
        ops["target_pe"] = 3
        ops["rem_off"] = [a + (k << 20) for k in range(4)] + [a + (4 << 20), 0, a + (5 << 20)]
        ops["loc_off"] = ops["rem_off"]
        ops["nbytes"] = [1 << 20] * 4 + [256, 0, 8]
        ops["ctx"] = [0] * 4 + [ctx_small] * 3
        b = w.batch(ops)
        raw = b.plan.cpu().numpy()
        ntiles = int(raw[:4].view(np.uint32)[0])
        recs = raw[256:256 + 64 * ntiles].reshape(ntiles, 64)
        last = recs[-1]
        return int(last[48:52].view(np.uint32)[0]), int(last[52:56].view(np.uint32)[0]), b

    dom, dep, b = plan(1)
    assert (dom, dep) == (4 + 2, 1)
    w.enqueue_batch(b); w.quiet(0)
    dom, dep, b = plan(0)
    assert (dom, dep) == (2, 5)
