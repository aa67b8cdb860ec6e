"""Neutral description of an op-batch workload (inputs only, no method arithmetic).

A `Program` names symmetric objects (by size), their per-PE initial contents and an
ordered list of one-sided ops that address `(object, byte offset)` pairs.  The CUDA
harness and the oracle harness each resolve object names to their OWN symmetric
offsets (their own allocators) and translate the op records to their OWN descriptor
formats, so the two sides share nothing but this input description.

Op vocabulary follows SURVEY.md section 8(b)/(c).
"""
from __future__ import annotations

import numpy as np

# neutral op kinds (each side maps these to its own opcode enum)
PUT, GET, PUT_SIGNAL, ATOMIC_ADD, ATOMIC_FETCH_ADD, ATOMIC_COMPARE_SWAP, \
    SIGNAL_WAIT_UNTIL, FENCE, QUIET, BARRIER_ALL = range(1, 11)
KIND_NAMES = {PUT: "PUT", GET: "GET", PUT_SIGNAL: "PUT_SIGNAL", ATOMIC_ADD: "ATOMIC_ADD",
              ATOMIC_FETCH_ADD: "ATOMIC_FETCH_ADD", ATOMIC_COMPARE_SWAP: "ATOMIC_COMPARE_SWAP",
              SIGNAL_WAIT_UNTIL: "SIGNAL_WAIT_UNTIL", FENCE: "FENCE", QUIET: "QUIET",
              BARRIER_ALL: "BARRIER_ALL"}
SIGNAL_SET, SIGNAL_ADD = 0, 1
CMP_EQ, CMP_NE, CMP_GT, CMP_GE, CMP_LT, CMP_LE = range(6)

NOBJ = -1

OP_DTYPE = np.dtype([
    ("kind", "u1"), ("sig_op", "u1"), ("cmp", "u1"), ("ctx", "u1"),
    ("initiator", "i4"), ("target", "i4"),
    ("rem_obj", "i4"), ("loc_obj", "i4"), ("sig_obj", "i4"),
    ("rem_off", "u8"), ("loc_off", "u8"), ("nbytes", "u8"),
    ("value", "u8"), ("cond", "u8"), ("sig_off", "u8"),
])

U64 = (1 << 64) - 1


class Program:
    """npes logical PEs, named symmetric objects, ordered op list."""

    def __init__(self, npes: int):
        self.npes = int(npes)
        self.obj_names: list[str] = []
        self.obj_bytes: list[int] = []
        self.init: dict[str, np.ndarray] = {}      # name -> uint8 [npes, nbytes]; absent = zero
        self._ops: list[tuple] = []
        self._arr: np.ndarray | None = None

    # ---- objects -------------------------------------------------------------------------
    def obj(self, name: str, nbytes: int, init: np.ndarray | None = None) -> int:
        assert name not in self.obj_names
        self.obj_names.append(name)
        self.obj_bytes.append(int(nbytes))
        if init is not None:
            a = np.ascontiguousarray(init).view(np.uint8).reshape(self.npes, -1)
            assert a.shape[1] == nbytes, (a.shape, nbytes)
            self.init[name] = a
        return len(self.obj_names) - 1

    def oid(self, name: str) -> int:
        return self.obj_names.index(name)

    # ---- ops -----------------------------------------------------------------------------
    def _add(self, kind, initiator, target=0, rem=(NOBJ, 0), loc=(NOBJ, 0), nbytes=0, value=0, cond=0,
             sig=(NOBJ, 0), sig_op=0, cmp=0, ctx=0):
        def o(x):
            return (self.oid(x[0]) if isinstance(x[0], str) else int(x[0]), int(x[1]))
        rem, loc, sig = o(rem), o(loc), o(sig)
        self._ops.append((kind, sig_op, cmp, ctx, initiator, target, rem[0], loc[0], sig[0],
                          rem[1], loc[1], nbytes, value & U64, cond & U64, sig[1]))
        self._arr = None

    def put(self, pe, target, dst, src, nbytes, ctx=0):
        self._add(PUT, pe, target, rem=dst, loc=src, nbytes=nbytes, ctx=ctx)

    def get(self, pe, target, dst, src, nbytes, ctx=0):
        self._add(GET, pe, target, rem=src, loc=dst, nbytes=nbytes, ctx=ctx)

    def put_signal(self, pe, target, dst, src, nbytes, sig, sig_value, sig_op=SIGNAL_SET, ctx=0):
        self._add(PUT_SIGNAL, pe, target, rem=dst, loc=src, nbytes=nbytes, sig=sig, value=sig_value,
                  sig_op=sig_op, ctx=ctx)

    def atomic_add(self, pe, target, dst, value, ctx=0):
        self._add(ATOMIC_ADD, pe, target, rem=dst, value=value, nbytes=8, ctx=ctx)

    def atomic_fetch_add(self, pe, target, dst, value, fetch, ctx=0):
        self._add(ATOMIC_FETCH_ADD, pe, target, rem=dst, loc=fetch, value=value, nbytes=8, ctx=ctx)

    def atomic_compare_swap(self, pe, target, dst, cond, value, fetch, ctx=0):
        self._add(ATOMIC_COMPARE_SWAP, pe, target, rem=dst, loc=fetch, value=value, cond=cond, nbytes=8, ctx=ctx)

    def signal_wait_until(self, pe, sig, cmp, value, ctx=0):
        self._add(SIGNAL_WAIT_UNTIL, pe, pe, loc=sig, cmp=cmp, value=value, ctx=ctx)

    def fence(self, pe, ctx=0):
        self._add(FENCE, pe, pe, ctx=ctx)

    def quiet(self, pe, ctx=0):
        self._add(QUIET, pe, pe, ctx=ctx)

    def barrier_all(self):
        self._add(BARRIER_ALL, 0, 0)

    @property
    def ops(self) -> np.ndarray:
        if self._arr is None:
            self._arr = np.array(self._ops, dtype=OP_DTYPE) if self._ops else np.zeros(0, dtype=OP_DTYPE)
        return self._arr

    def set_ops(self, arr: np.ndarray):
        """Install a vectorised op array directly (large generated batches)."""
        assert arr.dtype == OP_DTYPE
        self._arr = arr
        self._ops = []

    def fork(self) -> "Program":
        """Same objects (shared by reference), empty op list: one batch of a multi-batch workload."""
        q = Program(self.npes)
        q.obj_names, q.obj_bytes, q.init = self.obj_names, self.obj_bytes, self.init
        return q

    def __len__(self):
        return len(self.ops)
