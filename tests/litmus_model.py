"""Brute-force enumerator of the ordering model on tiny programs.

Independent of oracle/ and of the CUDA path: plain Python, word-granular memory, exhaustive DFS over
every schedule the ordering rules allow.  It pins the oracle's treatment of fence / quiet / signal /
barrier / atomics (the oracle's single schedule must land inside the reachable set, and the set must be a
singleton for determinate programs) and gives the GPU tests the set of legal outcomes for tiny programs.

Rules (put_signal per SURVEY.md reading 8):
  * each PE runs its program in order; a scheduler step either ADVANCES one PE past its next op or
    DELIVERS one pending remote update;
  * PUT / GET / ATOMIC_* / PUT_SIGNAL are non-blocking (reading 7): on issue they enter the initiator's
    pending set; delivery applies them atomically (PUT_SIGNAL = payload delivery, after which its signal
    update becomes a separately pending delivery);
  * FENCE by p: no op p issued after the fence may be delivered before every op p issued before it
    (strong reading: any target; per-target reading: same target only -- both are enumerable);
  * QUIET by p: p cannot advance until its pending set is empty;
  * SIGNAL_WAIT_UNTIL by p: p cannot advance until the comparison holds on p's own heap;
  * BARRIER_ALL: nobody advances past it until all PEs have arrived and all pending sets are empty;
  * end of batch: implicit quiet for every PE.

Program format: prog[p] = list of ops, each a tuple:
  ("put", t, dst, src)            heap[t][dst] = heap[p][src]            (one word)
  ("get", t, dst, src)            heap[p][dst] = heap[t][src]
  ("put_signal", t, dst, src, sig, val, "set"|"add")
  ("add", t, dst, v) / ("fadd", t, dst, v, fetch) / ("cas", t, dst, cond, v, fetch)
  ("wait", sig, cmp, v)  cmp in {"eq","ne","gt","ge","lt","le"}
  ("fence",) / ("quiet",) / ("barrier",)
Contexts (reading 31): any op may carry a trailing "@c" (c = context number,
default "@0").  A context is an independent stream of operations of its PE: PROGRAM ORDER, FENCE, QUIET and
SIGNAL_WAIT_UNTIL act within one (PE, context) pair only; BARRIER_ALL covers every context of every PE.  The
enumerator therefore runs one in-order program per (PE, context) domain; addresses still name PEs.
"""
from __future__ import annotations

M64 = (1 << 64) - 1
_CMP = {"eq": lambda a, b: a == b, "ne": lambda a, b: a != b, "gt": lambda a, b: a > b,
        "ge": lambda a, b: a >= b, "lt": lambda a, b: a < b, "le": lambda a, b: a <= b}
_NB = ("put", "get", "put_signal", "add", "fadd", "cas")


def _set(heaps, p, i, v):
    h = list(heaps)
    row = list(h[p])
    row[i] = v & M64
    h[p] = tuple(row)
    return tuple(h)


def split_ctx(op):
    """(op without its context tag, context number)"""
    if isinstance(op[-1], str) and op[-1].startswith("@"):
        return tuple(op[:-1]), int(op[-1][1:])
    return tuple(op), 0


def _domains(prog):
    """Split per-PE programs into per-(PE, context) in-order programs; a barrier is replicated into every domain of
    its PE.  Returns (owner PE of each domain, domain programs)."""
    owner, dprog = [], []
    for p, ops in enumerate(prog):
        tagged = [split_ctx(op) for op in ops]
        ctxs = sorted({c for op, c in tagged if op[0] != "barrier"}) or [0]
        for c in ctxs:
            owner.append(p)
            dprog.append([op for op, cc in tagged if op[0] == "barrier" or cc == c])
    return owner, dprog


def enumerate_outcomes(prog, init_heaps, per_target_fence: bool = False, limit: int = 2_000_000):
    """Return the set of reachable final heaps (tuple of per-PE tuples of words)."""
    owner, prog = _domains(prog)          # from here on "p" indexes a (PE, context) domain, owner[p] is its PE
    npes = len(prog)
    # fence_before[p][i] = number of fences among ops 0..i-1 of p (its "fence epoch")
    epoch = []
    for p in range(npes):
        e, row = 0, []
        for op in prog[p]:
            row.append(e)
            if op[0] == "fence":
                e += 1
        epoch.append(row)

    def deliverable(p, pend, item):
        i, stage = item
        tgt = prog[p][i][1]
        for (j, _s) in pend:
            if j < i and epoch[p][j] < epoch[p][i]:
                if not per_target_fence or prog[p][j][1] == tgt:
                    return False
        return True

    def deliver(heaps, d, item):
        i, stage = item
        op = prog[d][i]
        p = owner[d]                      # the initiating PE (local heap of gets / fetch slots / put sources)
        k = op[0]
        follow = None
        if k == "put":
            heaps = _set(heaps, op[1], op[2], heaps[p][op[3]])
        elif k == "get":
            heaps = _set(heaps, p, op[2], heaps[op[1]][op[3]])
        elif k == "put_signal":
            if stage == 0:
                heaps = _set(heaps, op[1], op[2], heaps[p][op[3]])
                follow = (i, 1)
            else:
                old = heaps[op[1]][op[4]]
                heaps = _set(heaps, op[1], op[4], op[5] if op[6] == "set" else old + op[5])
        elif k == "add":
            heaps = _set(heaps, op[1], op[2], heaps[op[1]][op[2]] + op[3])
        elif k == "fadd":
            old = heaps[op[1]][op[2]]
            heaps = _set(heaps, op[1], op[2], old + op[3])
            heaps = _set(heaps, p, op[4], old)
        elif k == "cas":
            old = heaps[op[1]][op[2]]
            if old == (op[3] & M64):
                heaps = _set(heaps, op[1], op[2], op[4])
            heaps = _set(heaps, p, op[5], old)
        else:
            raise ValueError(k)
        return heaps, follow

    finals = set()
    seen = set()
    init = (tuple(0 for _ in range(npes)), tuple(() for _ in range(npes)),
            tuple(tuple(w & M64 for w in h) for h in init_heaps))
    stack = [init]
    while stack:
        st = stack.pop()
        if st in seen:
            continue
        seen.add(st)
        if len(seen) > limit:
            raise RuntimeError("state space too large")
        pcs, pends, heaps = st
        moved = False
        # deliveries
        for p in range(npes):
            for item in pends[p]:
                if deliverable(p, pends[p], item):
                    h2, follow = deliver(heaps, p, item)
                    np_ = tuple(x for x in pends[p] if x != item) + ((follow,) if follow else ())
                    stack.append((pcs, pends[:p] + (tuple(sorted(np_)),) + pends[p + 1:], h2))
                    moved = True
        # advances
        at_barrier = [pcs[p] < len(prog[p]) and prog[p][pcs[p]][0] == "barrier" for p in range(npes)]
        for p in range(npes):
            if pcs[p] >= len(prog[p]):
                continue
            op = prog[p][pcs[p]]
            k = op[0]
            if k in _NB:
                np_ = tuple(sorted(pends[p] + ((pcs[p], 0),)))
                stack.append((pcs[:p] + (pcs[p] + 1,) + pcs[p + 1:], pends[:p] + (np_,) + pends[p + 1:], heaps))
                moved = True
            elif k == "fence":
                stack.append((pcs[:p] + (pcs[p] + 1,) + pcs[p + 1:], pends, heaps))
                moved = True
            elif k == "quiet":
                if not pends[p]:
                    stack.append((pcs[:p] + (pcs[p] + 1,) + pcs[p + 1:], pends, heaps))
                    moved = True
            elif k == "wait":
                if _CMP[op[2]](heaps[owner[p]][op[1]], op[3] & M64):
                    stack.append((pcs[:p] + (pcs[p] + 1,) + pcs[p + 1:], pends, heaps))
                    moved = True
            elif k == "barrier":
                if p == 0 and all(at_barrier) and not any(pends):
                    stack.append((tuple(pc + 1 for pc in pcs), pends, heaps))
                    moved = True
            else:
                raise ValueError(k)
        if not moved:
            done = all(pcs[p] >= len(prog[p]) for p in range(npes)) and not any(pends)
            if done:
                finals.add(heaps)
            else:
                # a deadlocked state (e.g. an unsatisfiable wait): report it as an outcome marker
                finals.add(("DEADLOCK", pcs))
    return finals


def to_spec_program(prog, init_heaps, order):
    """The same tiny program as a workloads.spec.Program (one 8-byte word per model word).

    `order` is a list of PE ids: the k-th entry emits the next op of that PE, giving the batch index
    order (the caller chooses one that is a legal sequential schedule)."""
    import numpy as np
    from workloads.spec import (CMP_EQ, CMP_GE, CMP_GT, CMP_LE, CMP_LT, CMP_NE, SIGNAL_ADD, SIGNAL_SET,
                                Program)
    cmpmap = {"eq": CMP_EQ, "ne": CMP_NE, "gt": CMP_GT, "ge": CMP_GE, "lt": CMP_LT, "le": CMP_LE}
    npes, nw = len(prog), len(init_heaps[0])
    sp = Program(npes)
    sp.obj("w", nw * 8, np.array(init_heaps, dtype=np.uint64))
    pcs = [0] * npes
    for p in order:
        op, c = split_ctx(prog[p][pcs[p]])
        pcs[p] += 1
        k = op[0]
        if k == "put":
            sp.put(p, op[1], ("w", op[2] * 8), ("w", op[3] * 8), 8, ctx=c)
        elif k == "get":
            sp.get(p, op[1], ("w", op[2] * 8), ("w", op[3] * 8), 8, ctx=c)
        elif k == "put_signal":
            sp.put_signal(p, op[1], ("w", op[2] * 8), ("w", op[3] * 8), 8, ("w", op[4] * 8), op[5],
                          SIGNAL_SET if op[6] == "set" else SIGNAL_ADD, ctx=c)
        elif k == "add":
            sp.atomic_add(p, op[1], ("w", op[2] * 8), op[3], ctx=c)
        elif k == "fadd":
            sp.atomic_fetch_add(p, op[1], ("w", op[2] * 8), op[3], ("w", op[4] * 8), ctx=c)
        elif k == "cas":
            sp.atomic_compare_swap(p, op[1], ("w", op[2] * 8), op[3], op[4], ("w", op[5] * 8), ctx=c)
        elif k == "wait":
            sp.signal_wait_until(p, ("w", op[1] * 8), cmpmap[op[2]], op[3], ctx=c)
        elif k == "fence":
            sp.fence(p, ctx=c)
        elif k == "quiet":
            sp.quiet(p, ctx=c)
        elif k == "barrier":
            if p == 0:
                sp.barrier_all()
        else:
            raise ValueError(k)
    assert all(pcs[p] == len(prog[p]) for p in range(npes)), "order does not cover the program"
    return sp
