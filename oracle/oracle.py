"""Python front-end of the CPU ORACLE (oracle/shmemg_oracle.c).  TEST INFRASTRUCTURE, NOT PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / `--impl reference` legs may import
this module.  It never imports the CUDA package, and the CUDA package never imports it.

`OracleWorld` owns N heaps as one numpy array `[npes, heap_bytes]` and a bump allocator that hands out
the same offset on every PE ("same size and allocation order").  Everything
else is a thin call into the C file, which follows SURVEY.md section 8(c) row by row.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "shmemg_oracle.c")
_SO = os.path.join(_HERE, "_oracle.so")
_lib = None

ERR_NAMES = {0: "OK", 1: "RANGE", 2: "WAIT_UNSATISFIED", 3: "OPCODE", 4: "ALIGN"}

# the oracle's own descriptor layout (mirrors orc_op_t in the C file; 72 bytes)
ORC_OP_DTYPE = np.dtype([
    ("opcode", "i4"), ("initiator", "i4"), ("target", "i4"), ("sig_op", "i4"), ("cmp", "i4"), ("_pad", "i4"),
    ("rem_off", "u8"), ("loc_off", "u8"), ("nbytes", "u8"), ("value", "u8"), ("cond", "u8"), ("sig_off", "u8"),
])


class OracleError(RuntimeError):
    pass


def build(force: bool = False) -> str:
    """Compile the oracle with the system C compiler (-O2, single-threaded by construction)."""
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        tmp = _SO + ".tmp%d" % os.getpid()
        subprocess.check_call(["gcc", "-O2", "-std=c11", "-shared", "-fPIC", "-o", tmp, _SRC])
        os.replace(tmp, _SO)
    return _SO


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        u64, vp, i = C.c_uint64, C.c_void_p, C.c_int
        L.orc_exec_batch.argtypes = [vp, i, u64, vp, u64, vp]
        L.orc_atomic_add_batch.argtypes = [vp, i, u64, u64, vp, vp, vp, u64]
        L.orc_atomic_fetch_add_batch.argtypes = [vp, i, u64, u64, vp, vp, vp, vp, u64]
        L.orc_atomic_compare_swap_batch.argtypes = [vp, i, u64, u64, vp, vp, vp, vp, vp, u64]
        L.orc_sum_reduce_f32.argtypes = [vp, i, u64, u64, u64, u64, vp]
        L.orc_sum_reduce_i64.argtypes = [vp, i, u64, u64, u64, u64]
        L.orc_fcollect.argtypes = [vp, i, u64, u64, u64, u64]
        L.orc_alltoall.argtypes = [vp, i, u64, u64, u64, u64]
        L.orc_alltoalls.argtypes = [vp, i, u64, u64, u64, u64, u64, u64, u64, u64, u64]
        L.orc_copy_spaces.argtypes = [vp, u64, vp, u64, i, i, u64, i, u64, u64]
        L.orc_broadcast.argtypes = [vp, i, u64, u64, u64, u64, i]
        L.orc_reduce.argtypes = [vp, i, u64, i, i, u64, u64, u64]
        L.orc_amo_batch.argtypes = [vp, i, u64, i, i, u64, vp, vp, vp, vp, u64]
        L.orc_amo_cswap_batch.argtypes = [vp, i, u64, i, u64, vp, vp, vp, vp, vp, u64]
        L.orc_ibput.argtypes = [vp, i, u64, u64, u64, u64, u64, u64, u64, i, i, i]
        L.orc_signal_test.argtypes = [vp, i, u64, u64, i, u64, i]
        L.orc_signal_test_vec.argtypes = [vp, i, u64, u64, u64, i, u64, i, vp]
        L.orc_signal_test_vec.restype = C.c_int64
        L.orc_team_fcollect.argtypes = [vp, i, u64, i, i, i, u64, u64, u64]
        L.orc_team_alltoall.argtypes = [vp, i, u64, i, i, i, u64, u64, u64]
        L.orc_team_broadcast.argtypes = [vp, i, u64, i, i, i, u64, u64, u64, i]
        L.orc_team_reduce.argtypes = [vp, i, u64, i, i, i, i, i, u64, u64, u64]
        L.orc_halo_delta.argtypes = [u64, u64, u64]
        L.orc_halo_delta.restype = C.c_double
        L.orc_halo_perturb.argtypes = [vp, u64, i, i, i, u64, u64]
        L.orc_halo_perturb.restype = None
        L.orc_halo_pack.argtypes = [vp, u64, i, vp]
        L.orc_halo_pack.restype = None
        L.orc_checksum64.argtypes = [vp, u64]
        L.orc_checksum64.restype = u64
        _lib = L
    return _lib


def _chk(rc: int, what: str, idx: int | None = None):
    if rc != 0:
        raise OracleError("%s: %s%s" % (what, ERR_NAMES.get(rc, rc), "" if idx is None else " at op %d" % idx))


def _u64arr(a) -> np.ndarray:
    a = np.ascontiguousarray(a)
    if a.dtype != np.uint64:
        a = a.astype(np.int64, copy=False).view(np.uint64) if a.dtype.kind == "i" and a.dtype.itemsize == 8 \
            else a.astype(np.uint64)
    return a


class OracleWorld:
    ALIGN = 256

    def __init__(self, npes: int, heap_bytes: int):
        self.npes = int(npes)
        self.heap_bytes = int(heap_bytes)
        self.heap = np.zeros((self.npes, self.heap_bytes), dtype=np.uint8)
        self._brk = 0
        self.objs: dict[str, tuple[int, int]] = {}

    # ---- symmetric allocation (a2): one offset valid on every PE ------------------------------
    def malloc(self, nbytes: int, name: str | None = None) -> int:
        off = (self._brk + self.ALIGN - 1) // self.ALIGN * self.ALIGN
        if off + nbytes > self.heap_bytes:
            raise OracleError("symmetric heap exhausted")
        self._brk = off + nbytes
        if name is not None:
            self.objs[name] = (off, nbytes)
        return off

    def view(self, off: int, nbytes: int, dtype=np.uint8) -> np.ndarray:
        """[npes, nbytes/itemsize] view of a symmetric object."""
        return self.heap[:, off:off + nbytes].view(dtype)

    def obj(self, name: str, dtype=np.uint8) -> np.ndarray:
        off, n = self.objs[name]
        return self.view(off, n, dtype)

    # ---- neutral Program -> oracle descriptors ---------------------------------------------------
    def load_program(self, prog):
        """Allocate the program's objects in order and install their initial contents."""
        for name, nb in zip(prog.obj_names, prog.obj_bytes):
            off = self.malloc(nb, name)
            if name in prog.init:
                self.heap[:, off:off + nb] = prog.init[name]

    def translate(self, prog) -> np.ndarray:
        ops = prog.ops
        base = np.array([self.objs[n][0] for n in prog.obj_names] + [0], dtype=np.uint64)  # [-1] -> 0
        out = np.zeros(len(ops), dtype=ORC_OP_DTYPE)
        out["opcode"] = ops["kind"]          # oracle opcodes 1..10, defined in the C file
        out["initiator"] = ops["initiator"]
        out["target"] = ops["target"]
        out["sig_op"] = ops["sig_op"]
        out["cmp"] = ops["cmp"]
        out["rem_off"] = base[ops["rem_obj"]] + ops["rem_off"]
        out["loc_off"] = base[ops["loc_obj"]] + ops["loc_off"]
        out["sig_off"] = base[ops["sig_obj"]] + ops["sig_off"]
        out["nbytes"] = ops["nbytes"]
        out["value"] = ops["value"]
        out["cond"] = ops["cond"]
        return out

    def exec_ops(self, orc_ops: np.ndarray):
        assert orc_ops.dtype == ORC_OP_DTYPE
        orc_ops = np.ascontiguousarray(orc_ops)
        err = C.c_uint64(0)
        rc = lib().orc_exec_batch(self.heap.ctypes.data, self.npes, self.heap_bytes, orc_ops.ctypes.data,
                                  len(orc_ops), C.byref(err))
        _chk(rc, "exec_batch", err.value)

    def run_program(self, prog):
        self.exec_ops(self.translate(prog))

    # ---- SoA AMO batches ------------------------------------------------------------------------
    def atomic_add_batch(self, sym_off, tgt_pe, idx, val):
        tgt_pe = np.ascontiguousarray(tgt_pe, dtype=np.int32)
        idx, val = _u64arr(idx), _u64arr(val)
        _chk(lib().orc_atomic_add_batch(self.heap.ctypes.data, self.npes, self.heap_bytes, sym_off,
                                        tgt_pe.ctypes.data, idx.ctypes.data, val.ctypes.data, len(idx)),
             "atomic_add_batch")

    def atomic_fetch_add_batch(self, sym_off, tgt_pe, idx, val) -> np.ndarray:
        tgt_pe = np.ascontiguousarray(tgt_pe, dtype=np.int32)
        idx, val = _u64arr(idx), _u64arr(val)
        fetched = np.empty(len(idx), dtype=np.uint64)
        _chk(lib().orc_atomic_fetch_add_batch(self.heap.ctypes.data, self.npes, self.heap_bytes, sym_off,
                                              tgt_pe.ctypes.data, idx.ctypes.data, val.ctypes.data,
                                              fetched.ctypes.data, len(idx)), "atomic_fetch_add_batch")
        return fetched

    def atomic_compare_swap_batch(self, sym_off, tgt_pe, idx, cond, val) -> np.ndarray:
        tgt_pe = np.ascontiguousarray(tgt_pe, dtype=np.int32)
        idx, cond, val = _u64arr(idx), _u64arr(cond), _u64arr(val)
        fetched = np.empty(len(idx), dtype=np.uint64)
        _chk(lib().orc_atomic_compare_swap_batch(self.heap.ctypes.data, self.npes, self.heap_bytes, sym_off,
                                                 tgt_pe.ctypes.data, idx.ctypes.data, cond.ctypes.data,
                                                 val.ctypes.data, fetched.ctypes.data, len(idx)),
             "atomic_compare_swap_batch")
        return fetched

    # ---- collectives ----------------------------------------------------------------------------
    def sum_reduce_f32(self, dst_off, src_off, nreduce, want_r64: bool = False):
        r64 = np.empty(nreduce, dtype=np.float64) if want_r64 else None
        _chk(lib().orc_sum_reduce_f32(self.heap.ctypes.data, self.npes, self.heap_bytes, dst_off, src_off,
                                      nreduce, r64.ctypes.data if want_r64 else None), "sum_reduce_f32")
        return r64

    def sum_reduce_i64(self, dst_off, src_off, nreduce):
        _chk(lib().orc_sum_reduce_i64(self.heap.ctypes.data, self.npes, self.heap_bytes, dst_off, src_off,
                                      nreduce), "sum_reduce_i64")

    def fcollect(self, dst_off, src_off, nbytes):
        _chk(lib().orc_fcollect(self.heap.ctypes.data, self.npes, self.heap_bytes, dst_off, src_off, nbytes),
             "fcollect")

    def alltoall(self, dst_off, src_off, nbytes):
        _chk(lib().orc_alltoall(self.heap.ctypes.data, self.npes, self.heap_bytes, dst_off, src_off, nbytes),
             "alltoall")


    # ---- NEXT-4: block-strided alltoall (FFT-style transposes), the CPU space of the two-space model -------------------
    def alltoalls(self, dst_off, src_off, dst_pe_stride, src_pe_stride, dst_block_stride, src_block_stride, block, nblocks):
        _chk(lib().orc_alltoalls(self.heap.ctypes.data, self.npes, self.heap_bytes, dst_off, src_off, dst_pe_stride,
                                 src_pe_stride, dst_block_stride, src_block_stride, block, nblocks), "alltoalls")

    def attach_cpu_space(self, cpu_heap_bytes: int):
        """The CPU half of the two-space model: a second array of npes windows with its own allocator."""
        self.cpu_heap_bytes = int(cpu_heap_bytes)
        self.cpu_heap = np.zeros((self.npes, self.cpu_heap_bytes), dtype=np.uint8)
        self._cpu_brk = 0

    def cpu_malloc(self, nbytes: int) -> int:
        off = (self._cpu_brk + self.ALIGN - 1) // self.ALIGN * self.ALIGN
        if off + nbytes > self.cpu_heap_bytes:
            raise OracleError("CPU symmetric heap exhausted")
        self._cpu_brk = off + nbytes
        return off

    def cpu_view(self, off: int, nbytes: int, dtype=np.uint8) -> np.ndarray:
        return self.cpu_heap[:, off:off + nbytes].view(dtype)

    def _space(self, space: int):
        return (self.heap, self.heap_bytes) if space == 0 else (self.cpu_heap, self.cpu_heap_bytes)

    def put_space(self, dst_space, dst_off, src_space, src_off, nbytes, pe, target):
        """heap[dst_space][target][dst_off : +n] = heap[src_space][pe][src_off : +n]; space 0 = GPU, 1 = CPU."""
        (dh, db), (sh, sb) = self._space(dst_space), self._space(src_space)
        _chk(lib().orc_copy_spaces(dh.ctypes.data, db, sh.ctypes.data, sb, self.npes, target, dst_off, pe, src_off, nbytes), "put_space")

    def get_space(self, dst_space, dst_off, src_space, src_off, nbytes, pe, target):
        """heap[dst_space][pe][dst_off : +n] = heap[src_space][target][src_off : +n]."""
        (dh, db), (sh, sb) = self._space(dst_space), self._space(src_space)
        _chk(lib().orc_copy_spaces(dh.ctypes.data, db, sh.ctypes.data, sb, self.npes, pe, dst_off, target, src_off, nbytes), "get_space")

    # ---- NEXT-2 surface: broadcast, general reductions, generic AMOs, block-strided put/get, test ----
    RED = {"sum": 0, "prod": 1, "min": 2, "max": 3, "and": 4, "or": 5, "xor": 6}
    DTYPE = {"f32": 0, "i64": 1, "i32": 2, "f64": 3}
    AMO = {"add": 0, "and": 1, "or": 2, "xor": 3, "swap": 4, "fetch": 5}

    def broadcast(self, dst_off, src_off, nbytes, root):
        _chk(lib().orc_broadcast(self.heap.ctypes.data, self.npes, self.heap_bytes, dst_off, src_off, nbytes, root),
             "broadcast")

    def reduce(self, op: str, dtype: str, dst_off, src_off, nreduce):
        _chk(lib().orc_reduce(self.heap.ctypes.data, self.npes, self.heap_bytes, self.RED[op], self.DTYPE[dtype],
                              dst_off, src_off, nreduce), "reduce")

    def amo_batch(self, op: str, width: int, sym_off, tgt_pe, idx, val=None, fetch: bool = False):
        tgt_pe = np.ascontiguousarray(tgt_pe, dtype=np.int32)
        idx = _u64arr(idx)
        val = None if val is None else _u64arr(val)
        fetched = np.empty(len(idx), dtype=np.uint64) if fetch else None
        _chk(lib().orc_amo_batch(self.heap.ctypes.data, self.npes, self.heap_bytes, self.AMO[op], width, sym_off,
                                 tgt_pe.ctypes.data, idx.ctypes.data, None if val is None else val.ctypes.data,
                                 fetched.ctypes.data if fetch else None, len(idx)), "amo_batch")
        return fetched

    def amo_cswap_batch(self, width: int, sym_off, tgt_pe, idx, cond, val) -> np.ndarray:
        tgt_pe = np.ascontiguousarray(tgt_pe, dtype=np.int32)
        idx, cond, val = _u64arr(idx), _u64arr(cond), _u64arr(val)
        fetched = np.empty(len(idx), dtype=np.uint64)
        _chk(lib().orc_amo_cswap_batch(self.heap.ctypes.data, self.npes, self.heap_bytes, width, sym_off, tgt_pe.ctypes.data,
                                       idx.ctypes.data, cond.ctypes.data, val.ctypes.data, fetched.ctypes.data, len(idx)),
             "amo_cswap_batch")
        return fetched

    def ibput(self, dst_off, src_off, dst_stride, src_stride, block, nblocks, pe, target):
        _chk(lib().orc_ibput(self.heap.ctypes.data, self.npes, self.heap_bytes, dst_off, src_off, dst_stride,
                             src_stride, block, nblocks, pe, target, 0), "ibput")

    def ibget(self, dst_off, src_off, dst_stride, src_stride, block, nblocks, pe, target):
        _chk(lib().orc_ibput(self.heap.ctypes.data, self.npes, self.heap_bytes, dst_off, src_off, dst_stride,
                             src_stride, block, nblocks, pe, target, 1), "ibget")

    def signal_test_vec(self, sig_off, nelems, cmp, value, pe) -> np.ndarray:
        """Ascending positions k < nelems with cmp(u64 heap[pe][sig_off + 8k], value): test_some; all = (len == nelems);
        any = the first entry."""
        idx = np.empty(max(nelems, 1), dtype=np.uint64)
        n = lib().orc_signal_test_vec(self.heap.ctypes.data, self.npes, self.heap_bytes, sig_off, nelems, cmp, value, pe,
                                      idx.ctypes.data)
        if n < 0:
            raise OracleError("signal_test_vec: bad argument")
        return idx[:n].copy()

    # ---- NEXT-3: collectives over a strided team (start, stride, size); ranks are team-relative ----
    def team_fcollect(self, team, dst_off, src_off, nbytes):
        _chk(lib().orc_team_fcollect(self.heap.ctypes.data, self.npes, self.heap_bytes, *team, dst_off, src_off, nbytes),
             "team_fcollect")

    def team_alltoall(self, team, dst_off, src_off, nbytes):
        _chk(lib().orc_team_alltoall(self.heap.ctypes.data, self.npes, self.heap_bytes, *team, dst_off, src_off, nbytes),
             "team_alltoall")

    def team_broadcast(self, team, dst_off, src_off, nbytes, root_rank):
        _chk(lib().orc_team_broadcast(self.heap.ctypes.data, self.npes, self.heap_bytes, *team, dst_off, src_off, nbytes,
                                      root_rank), "team_broadcast")

    def team_reduce(self, team, op: str, dtype: str, dst_off, src_off, nreduce):
        _chk(lib().orc_team_reduce(self.heap.ctypes.data, self.npes, self.heap_bytes, *team, self.RED[op],
                                   self.DTYPE[dtype], dst_off, src_off, nreduce), "team_reduce")

    def signal_test(self, sig_off, cmp, value, pe) -> bool:
        r = lib().orc_signal_test(self.heap.ctypes.data, self.npes, self.heap_bytes, sig_off, cmp, value, pe)
        if r < 0:
            raise OracleError("signal_test: bad argument")
        return bool(r)


# ---- NEXT-4 (iii): PE -> GPU placement ("direct GPU-GPU fabrics ... load-store fabrics") -----------
# The paper names the fabrics and fixes no placement; SURVEY 8(e) gives "PE p -> GPU p mod G".  Written out: with G shards,
# global PE g lives on shard g mod G, as that shard's local PE g div G (reading 42).  A sharded world computes the
# SAME thing as one world of all the PEs, so the oracle of every sharded operation is the existing routine on the global
# world; these functions only say which rows of the global heap a shard holds.
def shard_of(g: int, nshards: int) -> int:
    return g % nshards


def shard_local_index(g: int, nshards: int) -> int:
    return g // nshards


def shard_global_pe(shard: int, local: int, nshards: int) -> int:
    return local * nshards + shard


def shard_rows(ow: "OracleWorld", shard: int, nshards: int, off: int, nbytes: int, dtype=np.uint8) -> np.ndarray:
    """What shard `shard` holds of the symmetric range [off, off + nbytes): the rows of its PEs, in local-PE order."""
    rows = [g for g in range(ow.npes) if shard_of(g, nshards) == shard]
    rows.sort(key=lambda g: shard_local_index(g, nshards))
    return ow.view(off, nbytes, dtype)[rows]


# ---- halo application compute (config C2) ----------------------------------------------------------
def halo_delta(seed: int, rnd: int, gidx: int) -> float:
    return float(lib().orc_halo_delta(seed, rnd, gidx))


def halo_perturb(U: np.ndarray, B: int, pcoord, seed: int, rnd: int):
    assert U.dtype == np.float64 and U.flags["C_CONTIGUOUS"] and U.size == B ** 3
    lib().orc_halo_perturb(U.ctypes.data, B, pcoord[0], pcoord[1], pcoord[2], seed, rnd)


def halo_pack(U: np.ndarray, B: int, f: int, send: np.ndarray):
    assert send.dtype == np.float64 and send.flags["C_CONTIGUOUS"] and send.size == B * B
    lib().orc_halo_pack(U.ctypes.data, B, f, send.ctypes.data)


def checksum64(a: np.ndarray) -> int:
    a = np.ascontiguousarray(a)
    assert a.nbytes % 8 == 0
    return int(lib().orc_checksum64(a.ctypes.data, a.nbytes // 8))
