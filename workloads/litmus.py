"""Litmus programs run at scale: op lists whose batch index order is a valid
sequential schedule and whose final state is the same under every legal schedule, so a GPU run that
reorders across a fence / quiet / signal / barrier produces a state that differs from the oracle's.

Inputs only (op lists + seeded payloads); no method arithmetic.
"""
from __future__ import annotations

import numpy as np

from . import gen
from .spec import CMP_EQ, CMP_GE, SIGNAL_ADD, SIGNAL_SET, Program


def _payload(npes, nbytes, seed, stream):
    n8 = (nbytes + 7) // 8
    return np.ascontiguousarray(gen.u64(npes * n8, seed, stream).view(np.uint8).reshape(npes, n8 * 8)[:, :nbytes])


def mp_fence(npes: int = 16, rounds: int = 24, nbytes: int = 40000, seed: int = 11, lag: int = 2) -> Program:
    """MP+fence: p: PUT data->t; FENCE; PUT flag->t.   t: WAIT flag; GET data (local).  Must see new data.
    Consumers of round r are emitted after the producers of round r+lag (real overlap on the GPU)."""
    prog = Program(npes)
    prog.obj("src", rounds * nbytes, _payload(npes, rounds * nbytes, seed, 0))
    flagsrc = np.tile(np.arange(1, rounds + 1, dtype=np.uint64), (npes, 1))
    prog.obj("flagsrc", rounds * 8, flagsrc)
    prog.obj("data", rounds * nbytes)
    prog.obj("flag", rounds * 8)
    prog.obj("out", rounds * nbytes)

    def produce(r):
        for p in range(npes):
            t = (p + 1 + r % (npes - 1)) % npes
            prog.put(p, t, ("data", r * nbytes), ("src", r * nbytes), nbytes)
            prog.fence(p)
            prog.put(p, t, ("flag", r * 8), ("flagsrc", r * 8), 8)

    def consume(r):
        for t in range(npes):
            prog.signal_wait_until(t, ("flag", r * 8), CMP_EQ, r + 1)
            prog.get(t, t, ("out", r * nbytes), ("data", r * nbytes), nbytes)

    for r in range(rounds + lag):
        if r < rounds:
            produce(r)
        if r - lag >= 0:
            consume(r - lag)
    return prog


def mp_quiet_third_party(npes: int = 12, rounds: int = 16, nbytes: int = 24000, seed: int = 12) -> Program:
    """MP+quiet: p: PUT d->t1; PUT d->t2; QUIET; PUT flag->t3.  t3: WAIT flag; GET from t1; GET from t2.
    Distinguishes quiet (all targets complete) from a per-target fence."""
    assert npes >= 4
    prog = Program(npes)
    prog.obj("src", rounds * nbytes, _payload(npes, rounds * nbytes, seed, 0))
    prog.obj("flagsrc", rounds * 8, np.tile(np.arange(1, rounds + 1, dtype=np.uint64), (npes, 1)))
    prog.obj("data", rounds * nbytes)           # slot r on t1 and t2 written by exactly one p
    prog.obj("flag", rounds * 8)
    prog.obj("out", rounds * 2 * nbytes)
    for r in range(rounds):
        trip = []
        for p in range(npes):
            t1, t2, t3 = (p + 1) % npes, (p + 2) % npes, (p + 3) % npes
            # slot r of `data` on t1 is written by p (dist 1) AND by p-1 (dist 2): give them halves
            prog.put(p, t1, ("data", r * nbytes), ("src", r * nbytes), nbytes // 2)
            prog.put(p, t2, ("data", r * nbytes + nbytes // 2), ("src", r * nbytes + nbytes // 2), nbytes - nbytes // 2)
            prog.quiet(p)
            prog.put(p, t3, ("flag", r * 8), ("flagsrc", r * 8), 8)
            trip.append((t3, t1, t2))
        for (t3, t1, t2) in trip:
            prog.signal_wait_until(t3, ("flag", r * 8), CMP_EQ, r + 1)
            prog.get(t3, t1, ("out", (2 * r) * nbytes), ("data", r * nbytes), nbytes // 2)
            prog.get(t3, t2, ("out", (2 * r + 1) * nbytes), ("data", r * nbytes + nbytes // 2), nbytes - nbytes // 2)
    return prog


def put_signal_sizes(npes: int = 8, seed: int = 13,
                     sizes=(1, 2, 3, 7, 8, 15, 16, 17, 31, 33, 255, 256, 257, 1000, 4095, 4096, 4097, 65535,
                            65536, 65537, 300001, 1 << 20, (1 << 21) + 13)) -> Program:
    """put_signal with payloads from 1 B to 2 MiB at odd sizes and odd offsets; the waiter copies the whole
    payload after its wait.  Source/dest offsets cycle through all 16 relative misalignments."""
    prog = Program(npes)
    pad = 64
    tot = sum(s + pad for s in sizes) + 64
    prog.obj("src", tot, _payload(npes, tot, seed, 0))
    prog.obj("data", tot)
    prog.obj("out", tot)
    prog.obj("sig", len(sizes) * 8)
    off = 0
    for k, s in enumerate(sizes):
        so, do = off + (k * 5) % 16, off + (k * 11 + 3) % 16
        for p in range(npes):
            t = (p + 1 + k) % npes
            prog.put_signal(p, t, ("data", do), ("src", so), s, ("sig", k * 8), k + 1, SIGNAL_SET)
        for t in range(npes):
            prog.signal_wait_until(t, ("sig", k * 8), CMP_EQ, k + 1)
            prog.get(t, t, ("out", so), ("data", do), s)
        off += s + pad
    return prog


def signal_add_fanin(npes: int = 16, rounds: int = 8, nbytes: int = 9000, seed: int = 14) -> Program:
    """k = npes-1 senders each put_signal(ADD 1) their own slot on one target; the target waits GE k*(r+1)
    (the word accumulates over rounds) and then reads all k payloads."""
    prog = Program(npes)
    k = npes - 1
    prog.obj("src", rounds * nbytes, _payload(npes, rounds * nbytes, seed, 0))
    prog.obj("data", rounds * npes * nbytes)
    prog.obj("out", rounds * npes * nbytes)
    prog.obj("sig", 8)
    for r in range(rounds):
        for t in range(npes):
            for p in range(npes):
                if p != t:
                    prog.put_signal(p, t, ("data", (r * npes + p) * nbytes), ("src", r * nbytes), nbytes,
                                    ("sig", 0), 1, SIGNAL_ADD)
        for t in range(npes):
            prog.signal_wait_until(t, ("sig", 0), CMP_GE, k * (r + 1))
            for p in range(npes):
                if p != t:
                    prog.get(t, t, ("out", (r * npes + p) * nbytes), ("data", (r * npes + p) * nbytes), nbytes)
    return prog


def barrier_stamp(npes: int = 32, rounds: int = 40) -> Program:
    """Round r: every PE writes r into slot r&1 of its right neighbour; BARRIER_ALL; reads its own slot
    into log[r].  Every log entry must equal r (SURVEY.md 8(c) barrier row)."""
    prog = Program(npes)
    prog.obj("stamps", (rounds + 1) * 8, np.tile(np.arange(rounds + 1, dtype=np.uint64), (npes, 1)))
    prog.obj("slot", 16)
    prog.obj("log", (rounds + 1) * 8)
    for r in range(1, rounds + 1):
        for p in range(npes):
            prog.put(p, (p + 1) % npes, ("slot", (r & 1) * 8), ("stamps", r * 8), 8)
        prog.barrier_all()
        for p in range(npes):
            prog.get(p, p, ("log", r * 8), ("slot", (r & 1) * 8), 8)
    return prog


def random_amos(npes: int = 8, nwords: int = 64, n_ops: int = 20000, seed: int = 15) -> Program:
    """Random ATOMIC_ADD / FETCH_ADD / COMPARE_SWAP ops through the general batch path.
    Words [0, nwords/2) receive adds and fetch-adds; words [nwords/2, nwords) receive CAS(-1 -> op id + 1).
    Every fetching op owns a private fetch slot in its initiator's heap."""
    prog = Program(npes)
    init = np.zeros((npes, nwords), dtype=np.uint64)
    init[:, nwords // 2:] = np.uint64(0xFFFFFFFFFFFFFFFF)
    prog.obj("words", nwords * 8, init)
    prog.obj("fetch", n_ops * 8)
    kind = gen.uniform_i32(n_ops, 0, 2, seed, 0)
    tgt = gen.uniform_i32(n_ops, 0, npes - 1, seed, 1)
    word = gen.uniform_i32(n_ops, 0, nwords // 2 - 1, seed, 2)
    val = gen.uniform_i64(n_ops, 1, 1000, seed, 3)
    for i in range(n_ops):
        p = i % npes
        if kind[i] == 0:
            prog.atomic_add(p, int(tgt[i]), ("words", int(word[i]) * 8), int(val[i]))
        elif kind[i] == 1:
            prog.atomic_fetch_add(p, int(tgt[i]), ("words", int(word[i]) * 8), int(val[i]), ("fetch", i * 8))
        else:
            prog.atomic_compare_swap(p, int(tgt[i]), ("words", (nwords // 2 + int(word[i])) * 8),
                                     0xFFFFFFFFFFFFFFFF, i + 1, ("fetch", i * 8))
    return prog


def wait_after_wait(npes: int = 4, groups: int = 6, chain: int = 24, nbytes: int = 1 << 20, seed: int = 16) -> Program:
    """A later wait of a PE that is satisfied EARLIER than the PE's previous wait must not let the ops between them start.
    Per group g (three PEs c, e, l; consumer c):  e: PUT_SIGNAL -> c (sig_early), at once.   l: `chain` x (PUT to itself;
    QUIET), then PUT_SIGNAL data -> c (sig_late).   c: WAIT sig_late; GET data -> out; WAIT sig_early; GET early -> out2.
    An executor that lets the second wait complete (and be counted) before the first one is satisfied starts the first GET
    on stale data."""
    assert npes >= 3
    prog = Program(npes)
    prog.obj("src", groups * nbytes, _payload(npes, groups * nbytes, seed, 0))
    prog.obj("scratch", nbytes)
    prog.obj("data", groups * nbytes)
    prog.obj("early", groups * 64)
    prog.obj("out", groups * nbytes)
    prog.obj("out2", groups * 64)
    prog.obj("sig", groups * 16)
    for g in range(groups):
        c, e, l = g % npes, (g + 1) % npes, (g + 2) % npes
        prog.put_signal(e, c, ("early", g * 64), ("src", g * 64), 64, ("sig", g * 16 + 8), g + 1, SIGNAL_SET)
        for _ in range(chain):
            prog.put(l, l, ("scratch", 0), ("src", g * nbytes), nbytes)
            prog.quiet(l)
        prog.put_signal(l, c, ("data", g * nbytes), ("src", g * nbytes), nbytes, ("sig", g * 16), g + 1, SIGNAL_SET)
        prog.signal_wait_until(c, ("sig", g * 16), CMP_EQ, g + 1)
        prog.get(c, c, ("out", g * nbytes), ("data", g * nbytes), nbytes)
        prog.signal_wait_until(c, ("sig", g * 16 + 8), CMP_EQ, g + 1)
        prog.get(c, c, ("out2", g * 64), ("early", g * 64), 64)
    return prog


def two_contexts(npes: int = 8, rounds: int = 10, big: int = 1 << 20, small: int = 4096, seed: int = 17) -> Program:
    """Every PE drives two contexts.  Context 0: a bulk stream (PUT big -> neighbour; QUIET(ctx 0); PUT_SIGNAL flag0).
    Context 1: a latency chain (PUT small -> other neighbour; QUIET(ctx 1); PUT flag1) issued between the bulk ops.  Consumers
    wait on the flags (on the context that produced them) and copy the payloads.  The result is the same for every legal
    schedule; an executor that lets a QUIET of one context order NOTHING (or that mixes the domains up) breaks it."""
    prog = Program(npes)
    prog.obj("src", rounds * (big + small), _payload(npes, rounds * (big + small), seed, 0))
    prog.obj("flagsrc", rounds * 8, np.tile(np.arange(1, rounds + 1, dtype=np.uint64), (npes, 1)))
    prog.obj("bulk", rounds * big)
    prog.obj("chain", rounds * small)
    prog.obj("flag0", rounds * 8)
    prog.obj("flag1", rounds * 8)
    prog.obj("out", rounds * (big + small))
    for r in range(rounds):
        for p in range(npes):
            t0, t1 = (p + 1) % npes, (p + 3) % npes
            prog.put(p, t0, ("bulk", r * big), ("src", r * (big + small)), big, ctx=0)
            prog.put(p, t1, ("chain", r * small), ("src", r * (big + small) + big), small, ctx=1)
            prog.quiet(p, ctx=1)
            prog.put(p, t1, ("flag1", r * 8), ("flagsrc", r * 8), 8, ctx=1)
            prog.quiet(p, ctx=0)
            prog.put_signal(p, t0, ("flag0", r * 8), ("flagsrc", r * 8), 0, ("flag0", r * 8), r + 1, SIGNAL_SET, ctx=0)
        for t in range(npes):
            prog.signal_wait_until(t, ("flag1", r * 8), CMP_EQ, r + 1, ctx=1)
            prog.get(t, t, ("out", r * (big + small) + big), ("chain", r * small), small, ctx=1)
            prog.signal_wait_until(t, ("flag0", r * 8), CMP_EQ, r + 1, ctx=0)
            prog.get(t, t, ("out", r * (big + small)), ("bulk", r * big), big, ctx=0)
    return prog


def contexts_amos_waits(npes: int = 8, rounds: int = 12, seed: int = 18) -> Program:
    """Fetching AMOs and waits on contexts > 0 (fetch slots and wait words are in the initiating PE's window whatever the
    context).  Round r, PE p, context c = 1 + r % 3:  FETCH_ADD(+r+1) and COMPARE_SWAP(-1 -> id) on words that only p
    touches on its neighbour t (so the fetched values are the same under every legal schedule), QUIET(c), then ATOMIC_ADD 1 on
    t's flag word of the round.  t waits (on another context) for that flag and copies the two words."""
    prog = Program(npes)
    init = np.zeros((npes, rounds * 2), dtype=np.uint64)
    init[:, 1::2] = np.uint64(0xFFFFFFFFFFFFFFFF)
    init[:, 0::2] = gen.u64(npes * rounds, seed, 0).reshape(npes, rounds)
    prog.obj("words", rounds * 16, init)
    prog.obj("flag", rounds * 8)
    prog.obj("fetch", rounds * 16)
    prog.obj("out", rounds * 16)
    for r in range(rounds):
        c = 1 + r % 3
        for p in range(npes):
            t = (p + 1 + r % (npes - 1)) % npes
            prog.atomic_fetch_add(p, t, ("words", r * 16), r + 1, ("fetch", r * 16), ctx=c)
            prog.atomic_compare_swap(p, t, ("words", r * 16 + 8), 0xFFFFFFFFFFFFFFFF, 1000 * r + p, ("fetch", r * 16 + 8), ctx=c)
            prog.quiet(p, ctx=c)
            prog.atomic_add(p, t, ("flag", r * 8), 1, ctx=c)
        for t in range(npes):
            c2 = 1 + (r + 1) % 3
            prog.signal_wait_until(t, ("flag", r * 8), CMP_GE, 1, ctx=c2)
            prog.get(t, t, ("out", r * 16), ("words", r * 16), 16, ctx=c2)
    return prog
