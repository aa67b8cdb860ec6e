"""GPU parity of the DEVICE-INITIATED path (include/shmemg_device.cuh): the same neutral
programs the batch executor runs are executed by PE-agent thread blocks that call the `__device__` entry points, and
compared with the CPU oracle object by object (bit-exact), plus the schedule-independent invariants for fetching
atomics and the brute-force outcome sets for tiny programs."""
import numpy as np
import pytest

from gpu_common import DEV, assert_objects_equal, run_gpu_device, run_gpu_device_ctx, run_oracle
from invariants import check_compare_swap_claim, check_fetch_add
from litmus_model import enumerate_outcomes, to_spec_program
from paper_2607_08006_b200 import CAP, ERR, OP, OP_DTYPE, TEAM, ShmemgError, World
from test_gpu_batch import TINY
from workloads import configs, gen, litmus
from workloads.spec import Program

pytestmark = pytest.mark.gpu
M64 = (1 << 64) - 1


def test_capabilities_distinguish_the_device_path():
    """capability queries distinguish host-initiated GPU-aware from device-initiated support."""
    w = World(4, 4096, DEV)
    host, dev = w.query_capabilities(TEAM.WORLD), w.query_capabilities(TEAM.DEVICE_WORLD)
    assert dev & CAP.DEVICE_INITIATED and dev & CAP.DEVICE_BARRIER and dev & CAP.DEVICE_COLLECTIVES
    assert not host & CAP.DEVICE_COLLECTIVES
    assert not host & CAP.DEVICE_INITIATED and host & CAP.STREAM_TRIGGERED
    assert w.query_capabilities(TEAM.DEVICE_SHARED) == dev          # one GPU: shared == world (L357)


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
], ids=["mp_fence", "mp_fence_big", "mp_quiet3", "put_signal_sizes", "signal_add_fanin", "barrier_stamp",
        "barrier_stamp128", "wait_after_wait", "two_contexts"])
def test_litmus_programs_device_initiated_match_oracle(make):
    prog = make()
    w, ld = run_gpu_device(prog)
    assert_objects_equal(prog, ld, run_oracle(prog))


def test_random_put_get_unaligned_device_initiated():
    """Race-free random puts/gets, arbitrary sizes and alignments (every head/body/tail width of shmemg_dev_copy)."""
    npes, nops, slot = 6, 600, 5000
    rng = np.random.default_rng(5)
    prog = Program(npes)
    prog.obj("src", 40000, gen.u64(npes * 40000 // 8, 78).view(np.uint8).reshape(npes, 40000))
    prog.obj("dst", nops * slot)
    for k in range(nops):
        i, t = int(rng.integers(npes)), int(rng.integers(npes))
        n = int(rng.integers(0, 70)) if k % 3 == 0 else int(rng.integers(0, slot - 32))
        s, d = int(rng.integers(0, 40000 - n)), k * slot + int(rng.integers(0, 32))
        if k % 4 == 1:
            s = (s & ~15) + (d & 15)                                 # congruent mod 16: head + vector body + tail
        if k % 2:
            prog.put(i, t, ("dst", d), ("src", s), n)
        else:
            prog.get(i, t, ("dst", d), ("src", s), n)
    w, ld = run_gpu_device(prog)
    assert_objects_equal(prog, ld, run_oracle(prog))


def test_random_amos_device_initiated():
    prog = litmus.random_amos()
    w, ld = run_gpu_device(prog)
    ow = run_oracle(prog)
    ops = prog.ops
    nw = prog.obj_bytes[0] // 8
    words = ld.obj_numpy("words", np.uint64)
    assert np.array_equal(words[:, :nw // 2], ow.obj("words", np.uint64)[:, :nw // 2])     # add / fetch-add finals
    assert np.array_equal(words[:, nw // 2:] == M64, ow.obj("words", np.uint64)[:, nw // 2:] == M64)
    fetch = ld.obj_numpy("fetch", np.uint64)
    key = ops["target"].astype(np.int64) * nw + (ops["rem_off"] // 8).astype(np.int64)
    fa, ad, cs = ops["kind"] == 5, ops["kind"] == 4, ops["kind"] == 6
    fetched = fetch[ops["initiator"], np.arange(len(ops))]
    sel = fa & ~np.isin(key, np.unique(key[ad]))
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


@pytest.mark.parametrize("name", sorted(TINY))
def test_tiny_programs_device_initiated_land_in_outcome_set(name):
    """Truly concurrent PE agents: the final state must be one the ordering rules allow (brute-force enumeration)."""
    prog, init, order = TINY[name]
    allowed = enumerate_outcomes(prog, init)
    sp = to_spec_program(prog, init, order)
    for _ in range(5):
        w, ld = run_gpu_device(sp)
        got = tuple(tuple(int(x) for x in row) for row in ld.obj_numpy("w", np.uint64))
        assert got in allowed, (name, got)


def test_halo_rounds_device_initiated_match_oracle():
    """Config 2's exchange (put_signal + wait + consume) for 4 rounds at B = 32, device-initiated, vs the oracle."""
    h = configs.Halo(32)
    prog = h.program(with_consume=True, with_U=False)
    prog.init["send"] = gen.u64(8 * 6 * h.face_bytes // 8, 21).view(np.uint8).reshape(8, -1)
    rounds = [h.round_ops(prog, r, True) for r in range(1, 5)]
    w, ld = run_gpu_device(prog, batches=rounds)
    assert_objects_equal(prog, ld, run_oracle(prog, batches=rounds))


def test_device_exec_rejects_bad_descriptors_and_empty_list():
    w = World(2, 4096, DEV)
    w.device_exec_ops(np.zeros(0, dtype=OP_DTYPE))
    o = np.zeros(1, dtype=OP_DTYPE)
    o["opcode"], o["target_pe"], o["nbytes"] = OP.PUT, 2, 8
    with pytest.raises(ShmemgError) as e:
        w.device_exec_ops(o)
    assert e.value.code == ERR.PE


@pytest.mark.parametrize("B,rounds,split", [(16, 20, 7), (5, 9, 9), (2, 4, 1), (1, 3, 3), (256, 2, 2)])
def test_halo_persistent_device_initiated_matches_oracle(B, rounds, split):
    """Config 2 run by ONE persistent device-initiated kernel (no pack kernel, no send buffer, no kernel boundary between
    rounds): U, both ghost buffers and the signal words must be bit-identical to the oracle's perturb + pack + put_signal /
    wait rounds.  `split`: the rounds are run as two launches (first `split`, then the rest) to cover a restart."""
    from oracle import oracle as orc
    from paper_2607_08006_b200.loader import Loaded
    h = configs.Halo(B)
    prog = h.program(with_consume=False)
    hb = sum((b + 255) // 256 * 256 for b in prog.obj_bytes) + 4096
    w = World(8, hb, DEV)
    ld = Loaded(w, prog)
    ow = orc.OracleWorld(8, hb)
    ow.load_program(prog)
    U_off, ghost_off, sig_off = ld.off["U"][0], ld.off["ghost"][0], ld.off["sig"][0]
    w.app_halo_persistent(U_off, ghost_off, sig_off, B, h.seed, 1, split)
    if rounds > split:
        w.app_halo_persistent(U_off, ghost_off, sig_off, B, h.seed, split + 1, rounds - split)
    w.quiet(0)
    for r in range(1, rounds + 1):
        Uo, so = ow.obj("U", np.float64), ow.obj("send", np.float64).reshape(8, 6, B * B)
        for p in range(8):
            orc.halo_perturb(Uo[p], B, h.coord(p), h.seed, r)
            for f in range(6):
                orc.halo_pack(Uo[p], B, f, so[p, f])
        ow.run_program(h.round_ops(prog, r, False))
    assert_objects_equal(prog, ld, ow, names=["ghost", "sig"])
    assert np.array_equal(ld.obj_numpy("U", np.float64), ow.obj("U", np.float64))


# ---- device collectives (shmemg_dev_{sum_reduce,fcollect,alltoall,broadcast}_block) ----------------------
from oracle import oracle as orc                                       # noqa: E402
from paper_2607_08006_b200.binding import DEVCOLL, F32, F64, I32, I64   # noqa: E402
import torch                                                            # noqa: E402


def _worlds(npes, hb):
    return World(npes, hb, DEV), orc.OracleWorld(npes, hb)


@pytest.mark.parametrize("npes,n,off", [(8, 4096, 0), (128, 1 << 14, 0), (5, 1001, 4), (3, 7, 0), (16, 1, 8), (128, 100, 0)])
def test_device_sum_reduce_matches_oracle(npes, n, off):
    """fp32 (fp64 accumulation in PE order: bit-equal to the oracle's (float) of the fp64 sum), int64, int32, fp64; ragged
    counts, fewer elements than PEs, unaligned (to 16 B) offsets, in place."""
    w, ow = _worlds(npes, 16 * n + 8192)
    s, d = w.malloc(8 * n + 64) + off, w.malloc(8 * n + 64) + off
    os_, od = ow.malloc(8 * n + 64) + off, ow.malloc(8 * n + 64) + off
    xf = gen.normal_f32(npes * n, 31).reshape(npes, n)
    w.view(s, 4 * n, torch.float32).copy_(torch.from_numpy(xf)); ow.view(os_, 4 * n, np.float32)[:] = xf
    w.device_collective(DEVCOLL.SUM_REDUCE, d, s, n, dtype=F32); ow.sum_reduce_f32(od, os_, n); w.quiet(0)
    assert np.array_equal(w.view(d, 4 * n, torch.float32).cpu().numpy(), ow.view(od, 4 * n, np.float32))
    xi = gen.uniform_i64(npes * n, -(1 << 40), 1 << 40, 32).reshape(npes, n)
    o8 = off & ~7
    s8, d8, os8, od8 = s - off + o8, d - off + o8, os_ - off + o8, od - off + o8
    w.view(s8, 8 * n, torch.int64).copy_(torch.from_numpy(xi)); ow.view(os8, 8 * n, np.int64)[:] = xi
    w.device_collective(DEVCOLL.SUM_REDUCE, d8, s8, n, dtype=I64); ow.sum_reduce_i64(od8, os8, n); w.quiet(0)
    assert np.array_equal(w.view(d8, 8 * n, torch.int64).cpu().numpy(), ow.view(od8, 8 * n, np.int64))
    w.device_collective(DEVCOLL.SUM_REDUCE, s8, s8, n, dtype=I64); ow.sum_reduce_i64(os8, os8, n); w.quiet(0)     # in place
    assert np.array_equal(w.view(s8, 8 * n, torch.int64).cpu().numpy(), ow.view(os8, 8 * n, np.int64))
    for dt, name, tt, nt in ((I32, "i32", torch.int32, np.int32), (F64, "f64", torch.float64, np.float64)):
        esz = np.dtype(nt).itemsize
        x = (gen.uniform_i64(npes * n, -1000, 1000, 33).reshape(npes, n)).astype(nt)
        w.view(s8, esz * n, tt).copy_(torch.from_numpy(x)); ow.view(os8, esz * n, nt)[:] = x
        w.device_collective(DEVCOLL.SUM_REDUCE, d8, s8, n, dtype=dt); ow.reduce("sum", name, od8, os8, n); w.quiet(0)
        assert np.array_equal(w.view(d8, esz * n, tt).cpu().numpy(), ow.view(od8, esz * n, nt))


@pytest.mark.parametrize("npes,nb,off", [(8, 4096, 0), (64, 32768, 0), (7, 1001, 3), (128, 513, 0), (4, 1, 5)])
def test_device_fcollect_alltoall_broadcast_match_oracle(npes, nb, off):
    w, ow = _worlds(npes, 3 * npes * (nb + 16) + 8192)
    s, d = w.malloc(npes * nb + 64) + off, w.malloc(npes * nb + 64) + (off * 7) % 16
    os_, od = ow.malloc(npes * nb + 64) + off, ow.malloc(npes * nb + 64) + (off * 7) % 16
    pay = np.ascontiguousarray(gen.u64(npes * (npes * nb // 8 + 1), 41).view(np.uint8).reshape(npes, -1)[:, :npes * nb])
    w.view(s, npes * nb).copy_(torch.from_numpy(pay)); ow.view(os_, npes * nb)[:] = pay
    w.device_collective(DEVCOLL.ALLTOALL, d, s, nb); ow.alltoall(od, os_, nb); w.quiet(0)
    assert np.array_equal(w.view(d, npes * nb).cpu().numpy(), ow.view(od, npes * nb))
    w.device_collective(DEVCOLL.FCOLLECT, d, s, nb); ow.fcollect(od, os_, nb); w.quiet(0)
    assert np.array_equal(w.view(d, npes * nb).cpu().numpy(), ow.view(od, npes * nb))
    for root in (0, npes - 1):
        w.device_collective(DEVCOLL.BROADCAST, d, s, nb, root=root); ow.broadcast(od, os_, nb, root); w.quiet(0)
        assert np.array_equal(w.view(d, npes * nb).cpu().numpy(), ow.view(od, npes * nb))


def test_device_collective_argument_checks():
    w = World(4, 1 << 16, DEV)
    a, b = w.malloc(4096), w.malloc(4096)
    for kw, code in [(dict(kind=9, dest_off=b, source_off=a, n=8), ERR.ARG),
                     (dict(kind=DEVCOLL.SUM_REDUCE, dest_off=b, source_off=a, n=8, dtype=7), ERR.ARG),
                     (dict(kind=DEVCOLL.SUM_REDUCE, dest_off=b + 4, source_off=a, n=8, dtype=I64), ERR.ALIGN),
                     (dict(kind=DEVCOLL.ALLTOALL, dest_off=b, source_off=a, n=1 << 15), ERR.RANGE),
                     (dict(kind=DEVCOLL.FCOLLECT, dest_off=a + 64, source_off=a, n=256), ERR.OVERLAP),
                     (dict(kind=DEVCOLL.BROADCAST, dest_off=b, source_off=a, n=8, root=4), ERR.PE)]:
        with pytest.raises(ShmemgError) as e:
            w.device_collective(**kw)
        assert e.value.code == code, (kw, e.value)
    w.device_collective(DEVCOLL.FCOLLECT, b, a, 0)               # zero bytes: nothing enqueued


# ---- explicit device contexts and non-blocking operations (shmemg_ctx_create, shmemg_dev_*_nbi, shmemg_dev_ctx_*) ---------------
@pytest.mark.parametrize("make", [
    lambda: litmus.mp_fence(),
    lambda: litmus.mp_quiet_third_party(),
    lambda: litmus.put_signal_sizes(),
    lambda: litmus.signal_add_fanin(),
    lambda: litmus.barrier_stamp(),
    lambda: litmus.wait_after_wait(),
    lambda: litmus.two_contexts(),
    lambda: litmus.contexts_amos_waits(),
], ids=["mp_fence", "mp_quiet3", "put_signal_sizes", "signal_add_fanin", "barrier_stamp", "wait_after_wait", "two_contexts",
        "contexts_amos_waits"])
def test_litmus_programs_with_explicit_contexts_match_oracle(make):
    prog = make()
    w, ld = run_gpu_device_ctx(prog)
    assert_objects_equal(prog, ld, run_oracle(prog))
    nctx = int(prog.ops["ctx"].max()) + 1
    for k in range(prog.npes * nctx):                                # everything issued on a context has completed
        issued, completed = w.ctx_counters(w._ctx_handles, k)
        assert issued == completed
    ops = prog.ops
    nb = np.isin(ops["kind"], (1, 2, 3))                              # PUT, GET, PUT_SIGNAL are the queued operations
    for p in (0, prog.npes - 1):
        for c in range(nctx):
            assert w.ctx_counters(w._ctx_handles, p * nctx + c)[0] == int((nb & (ops["initiator"] == p) & (ops["ctx"] == c)).sum())


@pytest.mark.parametrize("name", sorted(TINY))
def test_tiny_programs_with_explicit_contexts_land_in_enumerated_outcome_set(name):
    prog, init, order = TINY[name]
    allowed = enumerate_outcomes(prog, init)
    sp = to_spec_program(prog, init, order)
    for _ in range(3):
        w, ld = run_gpu_device_ctx(sp)
        got = tuple(tuple(int(x) for x in row) for row in ld.obj_numpy("w", np.uint64))
        assert got in allowed, (name, got)


def test_wait_blocks_the_whole_pe_agent_in_the_device_interpreter():
    """Where the two execution paths differ (shmemg.h "Batch semantics"): in k_device_exec_ops_ctx a SIGNAL_WAIT_UNTIL blocks the
    PE's agent, as OpenSHMEM's shmem_wait_until blocks the calling PE, so an op of ANOTHER context behind the wait always sees
    the awaited data; the batch executor orders only the wait's own context (both outcomes are in the model's set, and the
    batch executor's result is checked against that set in test_tiny_programs_land_in_enumerated_outcome_set)."""
    prog, init, order = TINY["ctx_wait_then_forward_on_other_ctx"]
    assert {h[0][4] for h in enumerate_outcomes(prog, init)} == {0, 42}
    sp = to_spec_program(prog, init, order)
    for _ in range(5):
        w, ld = run_gpu_device_ctx(sp)
        assert int(ld.obj_numpy("w", np.uint64)[0][4]) == 42


def test_quiet_on_one_context_leaves_the_other_contexts_operations_pending():
    """PAPER L327 / L331 + reading 31: a context has its own completion counters and lives in device memory across kernels.
    Kernel A (its list is not quieted at the end): PE 0 issues a non-blocking put on context 0, another on context 1, and a
    QUIET on context 1.  Afterwards context 1 reads (1 issued, 1 completed) and its data has arrived; context 0 reads (1, 0)
    and its destination is untouched -- an outcome the brute-force model allows
    (test_litmus_model.py::test_contexts_are_independent_ordering_domains).  Kernel B: QUIET on context 0 completes it."""
    from gpu_common import heap_bytes_for
    from paper_2607_08006_b200.loader import Loaded
    prog = Program(2)
    prog.obj("w", 64, np.arange(16, dtype=np.uint64).reshape(2, 8))
    prog.put(0, 1, ("w", 0), ("w", 8), 8, ctx=0)
    prog.put(0, 1, ("w", 16), ("w", 24), 8, ctx=1)
    prog.quiet(0, ctx=1)
    w = World(2, heap_bytes_for(prog), DEV)
    ld = Loaded(w, prog)
    handles, dev = w.ctx_create_all(2, 8)
    w.device_exec_ops_ctx(ld.translate(prog), dev, 2, flags=1)        # SHMEMG_EXEC_LEAVE_PENDING
    assert w.ctx_counters(handles, 0) == (1, 0) and w.ctx_counters(handles, 1) == (1, 1)
    got = ld.obj_numpy("w", np.uint64)
    assert got[1, 2] == 3 and got[1, 0] == 8                          # ctx 1 delivered (word 3 of PE 0 = 3), ctx 0 still pending
    b = prog.fork()
    b.quiet(0, ctx=0)
    w.device_exec_ops_ctx(ld.translate(b), dev, 2, flags=1)
    assert w.ctx_counters(handles, 0) == (1, 1)
    assert_objects_equal(prog, ld, run_oracle(prog))
    assert w.ctx_counters(handles, 2) == (0, 0)
    caps = w.query_capabilities(TEAM.DEVICE_WORLD)
    assert caps & CAP.EXPLICIT_DEVICE_CTX and not w.query_capabilities(TEAM.WORLD) & CAP.EXPLICIT_DEVICE_CTX


def test_nbi_forms_on_a_stream():
    npes, n = 4, 50000
    w = World(npes, 4 * n + 4096, DEV)
    s, d, sig = w.malloc(n), w.malloc(n), w.calloc(1, 8)
    pay = gen.u64(npes * (n // 8 + 1), 9).view(np.uint8).reshape(npes, -1)[:, :n]
    w.view(s, n).copy_(torch.from_numpy(np.ascontiguousarray(pay))); w.view(d, n).zero_()
    w.put_nbi(d, s, n, 0, 1); w.get_nbi(d, s, n, 2, 3)
    w.put_signal_nbi(d, s, n - 3, sig, 7, 0, 1, 0)
    w.quiet(0)
    got = w.view(d, n).cpu().numpy()
    assert np.array_equal(got[1], pay[0]) and np.array_equal(got[2], pay[3]) and np.array_equal(got[0, :n - 3], pay[1, :n - 3])
    assert w.view(sig, 8, torch.int64).cpu().numpy()[0, 0] == 7
