"""Ordering rules pinned by brute force (CPU only).

tests/litmus_model.py enumerates EVERY schedule the paper's ordering rules allow on tiny programs
(PAPER.md L116, L126, L365-L369, L377-L390).  Here: (i) the enumerator itself shows the textbook litmus
outcomes (forbidden outcome absent with the fence, present without it); (ii) the oracle's single schedule
lands inside the reachable set, and that set is a singleton for every determinate program.
"""
import numpy as np
import pytest

from litmus_model import enumerate_outcomes, to_spec_program
from oracle import oracle as orc

M64 = (1 << 64) - 1


def oracle_heaps(prog, init, order):
    sp = to_spec_program(prog, init, order)
    w = orc.OracleWorld(sp.npes, 1024)
    w.load_program(sp)
    w.run_program(sp)
    return tuple(tuple(int(x) for x in row) for row in w.obj("w", np.uint64))


# words:            0=data 1=flag 2=src 3=one 4=out
INIT2 = [[0, 0, 42, 1, 0], [0, 0, 0, 0, 0]]


def test_mp_fence_forbids_stale_data_and_no_fence_allows_it():
    with_fence = [[("put", 1, 0, 2), ("fence",), ("put", 1, 1, 3)],
                  [("wait", 1, "eq", 1), ("get", 1, 4, 0)]]
    no_fence = [[("put", 1, 0, 2), ("put", 1, 1, 3)],
                [("wait", 1, "eq", 1), ("get", 1, 4, 0)]]
    out_f = enumerate_outcomes(with_fence, INIT2)
    out_n = enumerate_outcomes(no_fence, INIT2)
    assert {h[1][4] for h in out_f} == {42}                      # flag-new / data-old is unreachable
    assert {h[1][4] for h in out_n} == {0, 42}                   # ... and reachable without the fence
    assert len(out_f) == 1
    assert oracle_heaps(with_fence, INIT2, [0, 0, 0, 1, 1]) in out_f
    assert oracle_heaps(no_fence, INIT2, [0, 0, 1, 1]) in out_n
    # the per-target reading gives the same guarantee here (both puts go to PE 1)
    assert enumerate_outcomes(with_fence, INIT2, per_target_fence=True) == out_f


def test_atomicity_does_not_imply_ordering():
    """L365: 'Atomicity does not imply ordering. Programs must use fence/quiet when ordering is required.'"""
    init = [[0, 0, 0, 0, 0], [0, 0, 0, 0, 0]]
    no_fence = [[("add", 1, 0, 7), ("add", 1, 1, 1)], [("wait", 1, "ge", 1), ("get", 1, 4, 0)]]
    fenced = [[("add", 1, 0, 7), ("fence",), ("add", 1, 1, 1)], [("wait", 1, "ge", 1), ("get", 1, 4, 0)]]
    assert {h[1][4] for h in enumerate_outcomes(no_fence, init)} == {0, 7}
    out = enumerate_outcomes(fenced, init)
    assert {h[1][4] for h in out} == {7} and len(out) == 1
    assert oracle_heaps(fenced, init, [0, 0, 0, 1, 1]) in out


def test_quiet_completes_to_all_targets_but_per_target_fence_does_not():
    # PE0: put data->PE1; X; put flag->PE2.   PE2: wait flag; get data from PE1.
    init = [[0, 0, 42, 1, 0], [0] * 5, [0] * 5]
    def prog(x):
        return [[("put", 1, 0, 2), x, ("put", 2, 1, 3)], [], [("wait", 1, "eq", 1), ("get", 1, 4, 0)]]
    quiet = enumerate_outcomes(prog(("quiet",)), init)
    assert {h[2][4] for h in quiet} == {42} and len(quiet) == 1
    assert enumerate_outcomes(prog(("quiet",)), init, per_target_fence=True) == quiet
    strong = enumerate_outcomes(prog(("fence",)), init)
    assert {h[2][4] for h in strong} == {42}                    # the strong fence reading the GPU path implements
    weak = enumerate_outcomes(prog(("fence",)), init, per_target_fence=True)
    assert {h[2][4] for h in weak} == {0, 42}                   # classic per-target fence: third party may see old data
    assert oracle_heaps(prog(("quiet",)), init, [0, 0, 0, 2, 2]) in quiet


def test_put_signal_signal_never_precedes_payload():
    prog = [[("put_signal", 1, 0, 2, 1, 9, "set")], [("wait", 1, "eq", 9), ("get", 1, 4, 0)]]
    out = enumerate_outcomes(prog, INIT2)
    assert len(out) == 1 and next(iter(out))[1][4] == 42
    assert oracle_heaps(prog, INIT2, [0, 1, 1]) in out
    # signal ADD fan-in from two senders
    init = [[0, 0, 5, 0, 0, 0], [0, 0, 6, 0, 0, 0], [0, 0, 0, 0, 0, 0]]
    fan = [[("put_signal", 2, 0, 2, 1, 1, "add")], [("put_signal", 2, 3, 2, 1, 1, "add")],
           [("wait", 1, "ge", 2), ("get", 2, 4, 0), ("get", 2, 5, 3)]]
    out = enumerate_outcomes(fan, init)
    assert len(out) == 1 and next(iter(out))[2][4:6] == (5, 6)
    assert oracle_heaps(fan, init, [0, 1, 2, 2, 2]) in out


def test_quiet_then_read_back_and_missing_quiet():
    init = [[0, 0, 42, 0, 0], [0] * 5]
    q = [[("put", 1, 0, 2), ("quiet",), ("get", 1, 4, 0)], []]
    nq = [[("put", 1, 0, 2), ("get", 1, 4, 0)], []]
    out = enumerate_outcomes(q, init)
    assert len(out) == 1 and next(iter(out))[0][4] == 42
    assert {h[0][4] for h in enumerate_outcomes(nq, init)} == {0, 42}
    assert oracle_heaps(q, init, [0, 0, 0]) in out
    # fence also orders a get after a put in the strong reading the GPU path implements (reading 5)
    f = [[("put", 1, 0, 2), ("fence",), ("get", 1, 4, 0)], []]
    assert {h[0][4] for h in enumerate_outcomes(f, init)} == {42}


def test_fetch_add_linearisations_and_cas_single_winner():
    init = [[0, 0], [0, 0]]
    fa = [[("fadd", 1, 0, 2, 1)], [("fadd", 1, 0, 3, 1)]]
    out = enumerate_outcomes(fa, init)
    assert {(h[0][1], h[1][1], h[1][0]) for h in out} == {(0, 2, 5), (3, 0, 5)}
    assert oracle_heaps(fa, init, [0, 1]) in out and oracle_heaps(fa, init, [1, 0]) in out
    initc = [[M64, 0], [M64, 0]]
    cas = [[("cas", 1, 0, M64, 100, 1)], [("cas", 1, 0, M64, 200, 1)]]
    out = enumerate_outcomes(cas, initc)
    assert {(h[1][0], h[0][1], h[1][1]) for h in out} == {(100, M64, 100), (200, 200, M64)}
    assert oracle_heaps(cas, initc, [0, 1]) in out


def test_barrier_all_completes_everything_before_it():
    init = [[0, 0, 42, 0, 0], [0, 0, 43, 0, 0]]
    prog = [[("put", 1, 0, 2), ("barrier",), ("get", 0, 4, 0)],
            [("put", 0, 0, 2), ("barrier",), ("get", 1, 4, 0)]]
    out = enumerate_outcomes(prog, init)
    assert len(out) == 1
    h = next(iter(out))
    assert (h[0][4], h[1][4]) == (43, 42)
    assert oracle_heaps(prog, init, [0, 1, 0, 1, 0, 1]) in out
    nob = [[("put", 1, 0, 2), ("get", 0, 4, 0)], [("put", 0, 0, 2), ("get", 1, 4, 0)]]
    assert len(enumerate_outcomes(nob, init)) == 4


def test_unsatisfiable_wait_is_reported_as_deadlock():
    out = enumerate_outcomes([[("wait", 0, "eq", 1)], []], [[0], [0]])
    assert all(h[0] == "DEADLOCK" for h in out)


@pytest.mark.parametrize("seed", range(6))
def test_oracle_inside_reachable_set_random_programs(seed):
    """Random 2-PE programs (<= 4 ops per PE, no waits): the oracle's result for several legal batch orders
    is always a member of the enumerated set."""
    rng = np.random.default_rng(seed)
    nw = 4
    init = [[int(x) for x in rng.integers(1, 50, nw)] for _ in range(2)]
    prog = []
    for p in range(2):
        ops = []
        for _ in range(int(rng.integers(2, 5))):
            k = int(rng.integers(0, 7))
            t, a, b = int(rng.integers(0, 2)), int(rng.integers(0, nw)), int(rng.integers(0, nw))
            if k == 0:
                ops.append(("put", t, a, b))
            elif k == 1:
                ops.append(("get", t, a, b))
            elif k == 2:
                ops.append(("add", t, a, int(rng.integers(1, 9))))
            elif k == 3:
                ops.append(("fadd", t, a, int(rng.integers(1, 9)), b))
            elif k == 4:
                ops.append(("fence",))
            elif k == 5:
                ops.append(("quiet",))
            else:
                ops.append(("put_signal", t, a, b, (a + 1) % nw, 3, "add"))
        prog.append(ops)
    out = enumerate_outcomes(prog, init)
    n0, n1 = len(prog[0]), len(prog[1])
    shuffled = [0] * n0 + [1] * n1
    rng.shuffle(shuffled)            # per-PE op order is kept: `order` only says whose turn it is
    for order in ([0] * n0 + [1] * n1, [1] * n1 + [0] * n0, list(shuffled)):
        assert oracle_heaps(prog, init, order) in out


def test_contexts_are_independent_ordering_domains():
    """PAPER L124-L130 / L327, reading 31: fence / quiet / wait act within one (PE, context) pair.  A QUIET (or
    FENCE) on context 1 does not complete (order) the PE's pending put on context 0; the same program on one context does."""
    init = [[0, 0, 42, 1, 0, 7], [0] * 6]
    #            PE0: data put on ctx A; small put + X + flag put on ctx B.   PE1: wait flag; read data.
    def prog(a, b, x):
        return [[("put", 1, 0, 2, a), ("put", 1, 5, 5, b), (x, b), ("put", 1, 1, 3, b)],
                [("wait", 1, "eq", 1), ("get", 1, 4, 0)]]
    for x in ("quiet", "fence"):
        two = enumerate_outcomes(prog("@0", "@1", x), init)
        assert {h[1][4] for h in two} == {0, 42}                # ctx 0's put may still be pending behind ctx 1's marker
        assert {h[1][5] for h in two} == {7}                    # ... but ctx 1's own earlier put is ordered before the flag
        one = enumerate_outcomes(prog("@0", "@0", x), init)
        assert {h[1][4] for h in one} == {42} and len(one) == 1
        same = enumerate_outcomes(prog("@1", "@1", x), init)    # the context number itself means nothing
        assert same == one
        assert oracle_heaps(prog("@0", "@1", x), init, [0, 0, 0, 0, 1, 1]) in two
    # a wait blocks only its own context's stream: the ctx-0 put of PE1 may be delivered before PE1's ctx-1 wait returns
    init2 = [[0, 0, 42, 1, 0, 0], [0, 0, 43, 0, 0, 0]]
    w = [[("get", 1, 4, 0), ("quiet",), ("put", 1, 1, 3)],                     # PE0 reads PE1's word 0, then raises the flag
         [("wait", 1, "eq", 1, "@1"), ("put", 1, 0, 2, "@1"), ("put", 1, 5, 2, "@0")]]
    out = enumerate_outcomes(w, init2)
    assert {h[0][4] for h in out} == {0}                        # the ctx-1 put follows the wait: PE0 always read the old word
    assert {h[1][0] for h in out} == {43} and {h[1][5] for h in out} == {43}
    assert oracle_heaps(w, init2, [0, 0, 0, 1, 1, 1]) in out


def test_wait_orders_only_its_own_context_in_a_batch():
    """The batch contract of shmemg.h: SIGNAL_WAIT_UNTIL with ctx = c orders the later ops of (PE, c) only.  PE1 waits for the
    flag on context 0 and forwards the received word to PE0 on context 1: the forward may carry the old word (0) or the new one
    (42).  With a second wait on the forwarding context only 42 is left.  (The device-initiated interpreter blocks the whole PE
    at a wait and always produces 42, an element of both sets.)"""
    init = [[0, 0, 42, 1, 0], [0] * 5]
    send = [("put", 1, 0, 2), ("fence",), ("put", 1, 1, 3)]
    weak = enumerate_outcomes([send, [("wait", 1, "eq", 1, "@0"), ("put", 0, 4, 0, "@1")]], init)
    assert {h[0][4] for h in weak} == {0, 42}
    both = enumerate_outcomes([send, [("wait", 1, "eq", 1, "@0"), ("wait", 1, "eq", 1, "@1"), ("put", 0, 4, 0, "@1")]], init)
    assert {h[0][4] for h in both} == {42}
    same_ctx = enumerate_outcomes([send, [("wait", 1, "eq", 1, "@1"), ("put", 0, 4, 0, "@1")]], init)
    assert {h[0][4] for h in same_ctx} == {42}


def test_barrier_covers_every_context():
    init = [[0, 0, 42, 0, 0], [0, 0, 43, 0, 0]]
    prog = [[("put", 1, 0, 2, "@2"), ("barrier",), ("get", 0, 4, 0, "@1")],
            [("put", 0, 0, 2, "@1"), ("barrier",), ("get", 1, 4, 0)]]
    out = enumerate_outcomes(prog, init)
    assert len(out) == 1
    h = next(iter(out))
    assert (h[0][4], h[1][4]) == (43, 42)
    assert oracle_heaps(prog, init, [0, 1, 0, 1, 0, 1]) in out
