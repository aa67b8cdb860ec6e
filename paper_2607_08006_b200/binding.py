"""ctypes binding of include/shmemg.h, include/shmemg_app.h and include/shmemg_probe.h (same names, marshalling only)."""
from __future__ import annotations

import ctypes as C
import os

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libshmemg.so")


class ShmemgError(RuntimeError):
    def __init__(self, code: int, what: str, detail: str = ""):
        self.code = code
        super().__init__("%s: %s%s" % (what, ERR.name(code), (" (%s)" % detail) if detail else ""))


class ERR:
    OK, ARG, PE, RANGE, ALIGN, NOMEM, CUDA, OVERLAP, NODEVICE = 0, -1, -2, -3, -4, -5, -6, -7, -8

    @staticmethod
    def name(code):
        for k, v in vars(ERR).items():
            if k.isupper() and v == code:
                return "SHMEMG_ERR_" + k if code else "SHMEMG_OK"
        return str(code)


class OP:
    PUT, GET, PUT_SIGNAL, ATOMIC_ADD, ATOMIC_FETCH_ADD, ATOMIC_COMPARE_SWAP, SIGNAL_WAIT_UNTIL, FENCE, QUIET, \
        BARRIER_ALL = range(1, 11)


class SIGNAL:
    SET, ADD = 0, 1


class CMP:
    EQ, NE, GT, GE, LT, LE = range(6)


class TEAM:
    WORLD, DEVICE_WORLD, DEVICE_SHARED = 0, 1, 2


class CAP:
    GPU_HEAP_PRESENT = 1 << 0
    DEFAULT_HEAP_IS_GPU = 1 << 1
    HOST_INITIATED_GPU_BUFFERS = 1 << 2
    STREAM_TRIGGERED = 1 << 3
    DEVICE_INITIATED = 1 << 4
    DEVICE_COLLECTIVES = 1 << 5
    EXPLICIT_DEVICE_CTX = 1 << 6
    PTR_DEVICE_ACCESSIBLE = 1 << 7
    PTR_HOST_ACCESSIBLE = 1 << 8
    PROGRESS_GPU_ONLY = 1 << 9
    PATH_DIRECT = 1 << 10
    ATOMICS_64 = 1 << 11
    STREAM_COLLECTIVES = 1 << 12
    DEVICE_BARRIER = 1 << 13
    CPU_HEAP_PRESENT = 1 << 14
    PEER_SHARDS = 1 << 15


F32, I64, I32, F64 = 0, 1, 2, 3


class RED:
    SUM, PROD, MIN, MAX, AND, OR, XOR = range(7)


class AMO:
    ADD, AND, OR, XOR, SWAP, FETCH = range(6)


class DEVCOLL:
    SUM_REDUCE, FCOLLECT, ALLTOALL, BROADCAST = range(4)


AMO_WARP_AGGREGATE = 1
AMO_TEST_BEFORE_SWAP = 2
AMO_HOT_AGGREGATE = 4
STATIC_MAX_OPS = 1 << 22                 # SHMEMG_STATIC_MAX_OPS
AMO_THEN_BARRIER = 8
NO_STAMP = (1 << 64) - 1

# shmemg_op_t, 64 bytes
OP_DTYPE = np.dtype([
    ("opcode", "u1"), ("sig_op", "u1"), ("cmp", "u1"), ("ctx", "u1"),
    ("initiator_pe", "i4"), ("target_pe", "i4"), ("reserved1", "u4"),
    ("rem_off", "u8"), ("loc_off", "u8"), ("nbytes", "u8"), ("value", "u8"), ("cond", "u8"), ("sig_off", "u8"),
])
assert OP_DTYPE.itemsize == 64

# every symbol include/shmemg.h and include/shmemg_app.h declare: name -> (restype, argtypes)
_vp, _u64, _sz, _i, _u32 = C.c_void_p, C.c_uint64, C.c_size_t, C.c_int, C.c_uint32
SYMBOLS = {
    "shmemg_slab_bytes_required": (_sz, [_i, _sz]),
    "shmemg_init": (_i, [_i, _sz, _vp, _sz, C.POINTER(_vp)]),
    "shmemg_finalize": (_i, [_vp]),
    "shmemg_n_pes": (_i, [_vp]),
    "shmemg_heap_bytes": (_sz, [_vp]),
    "shmemg_heap_stride": (_sz, [_vp]),
    "shmemg_last_cuda_error": (C.c_char_p, [_vp]),
    "shmem_query_capabilities": (_i, [_vp, _i, C.POINTER(_u64)]),
    "shmemg_malloc": (_i, [_vp, _sz, C.POINTER(_u64)]),
    "shmemg_calloc": (_i, [_vp, _sz, _sz, C.POINTER(_u64), _vp]),
    "shmemg_align": (_i, [_vp, _sz, _sz, C.POINTER(_u64)]),
    "shmemg_free": (_i, [_vp, _u64]),
    "shmemg_ptr": (_vp, [_vp, _u64, _i]),
    "shmemg_heap_write_on_stream": (_i, [_vp, _i, _u64, _vp, _sz, _vp]),
    "shmemg_heap_read_on_stream": (_i, [_vp, _i, _vp, _u64, _sz, _vp]),
    "shmemg_batch_plan_bytes": (_sz, [_vp, _vp, _sz]),
    "shmemg_batch_create": (_i, [_vp, _vp, _sz, _vp, _sz, _vp, C.POINTER(_vp), C.POINTER(_sz)]),
    "shmemg_batch_destroy": (_i, [_vp]),
    "shmemg_batch_launches": (_i, [_vp]),
    "shmemg_batch_enqueue_on_stream": (_i, [_vp, _vp, _vp]),
    "shmemg_set_dependent_launch": (_i, [_vp, _i]),
    "shmemg_batch_work_bytes": (_sz, [_vp, _sz, _u64]),
    "shmemg_enqueue_batch": (_i, [_vp, _vp, _sz, _vp]),
    "shmemg_enqueue_batch_ws": (_i, [_vp, _vp, _sz, _vp, _sz, _vp]),
    "shmemg_batch_status": (_i, [_vp, _vp, _vp, C.POINTER(_i), C.POINTER(_sz)]),
    "shmemg_shard_of": (_i, [_i, _i]),
    "shmemg_shard_local_index": (_i, [_i, _i]),
    "shmemg_shard_global_pe": (_i, [_i, _i, _i]),
    "shmemg_shard_init": (_i, [_vp, _i, _i]),
    "shmemg_shard_export": (_i, [_vp, _vp, C.POINTER(_u64)]),
    "shmemg_shard_attach_ipc": (_i, [_vp, _i, _vp, _u64]),
    "shmemg_shard_attach_ptr": (_i, [_vp, _i, _vp]),
    "shmemg_shard_global_npes": (_i, [_vp]),
    "shmemg_gput_on_stream": (_i, [_vp, _u64, _u64, _sz, _i, _i, _vp]),
    "shmemg_gget_on_stream": (_i, [_vp, _u64, _u64, _sz, _i, _i, _vp]),
    "shmemg_gput_signal_on_stream": (_i, [_vp, _u64, _u64, _sz, _u64, _u64, _i, _i, _i, _vp]),
    "shmemg_gsignal_wait_until_on_stream": (_i, [_vp, _u64, _i, _u64, _i, _vp]),
    "shmemg_gatomic_batch_on_stream": (_i, [_vp, _i, _u64, _vp, _vp, _i, _vp, _u64, _vp, _u64, _vp, _sz, _vp]),
    "shmemg_galltoall_on_stream": (_i, [_vp, _u64, _u64, _sz, _vp]),
    "shmemg_gfcollect_on_stream": (_i, [_vp, _u64, _u64, _sz, _vp]),
    "shmemg_gsum_reduce_on_stream": (_i, [_vp, _i, _u64, _u64, _sz, _vp]),
    "shmemg_gbarrier_all_on_stream": (_i, [_vp, _vp]),
    "shmemg_put_on_stream": (_i, [_vp, _u64, _u64, _sz, _i, _i, _vp]),
    "shmemg_get_on_stream": (_i, [_vp, _u64, _u64, _sz, _i, _i, _vp]),
    "shmemg_put_signal_on_stream": (_i, [_vp, _u64, _u64, _sz, _u64, _u64, _i, _i, _i, _vp]),
    "shmemg_signal_wait_until_on_stream": (_i, [_vp, _u64, _i, _u64, _i, _vp]),
    "shmemg_fence_on_stream": (_i, [_vp, _i, _vp]),
    "shmemg_quiet_on_stream": (_i, [_vp, _i, _vp]),
    "shmemg_quiet": (_i, [_vp, _i, _vp]),
    "shmemg_amo_scratch_bytes": (_sz, [_vp, _sz]),
    "shmemg_set_scratch": (_i, [_vp, _vp, _sz]),
    "shmemg_amo_last_path": (_i, [_vp]),
    "shmemg_atomic_add_batch_on_stream": (_i, [_vp, _u64, _vp, _vp, _i, _vp, _u64, _sz, _u32, _vp]),
    "shmemg_atomic_fetch_add_batch_on_stream": (_i, [_vp, _u64, _vp, _vp, _i, _vp, _u64, _vp, _sz, _u32, _vp]),
    "shmemg_atomic_fetch_add_batch_static_on_stream": (_i, [_vp, _u64, _vp, _vp, _i, _u64, _vp, _sz, _u32, _vp, C.POINTER(_i)]),
    "shmemg_atomic_compare_swap_batch_on_stream": (_i, [_vp, _u64, _vp, _vp, _i, _vp, _u64, _vp, _u64, _vp, _sz, _u32, _vp]),
    "shmemg_sum_reduce_on_stream": (_i, [_vp, _i, _u64, _u64, _sz, _vp]),
    "shmemg_reduce_on_stream": (_i, [_vp, _i, _i, _u64, _u64, _sz, _vp]),
    "shmemg_broadcast_on_stream": (_i, [_vp, _u64, _u64, _sz, _i, _vp]),
    "shmemg_atomic_op_batch_on_stream": (_i, [_vp, _i, _i, _u64, _vp, _vp, _i, _vp, _u64, _vp, _sz, _vp]),
    "shmemg_atomic_cswap_op_batch_on_stream": (_i, [_vp, _i, _u64, _vp, _vp, _i, _vp, _u64, _vp, _u64, _vp, _sz, _vp]),
    "shmemg_amo_check_batch_on_stream": (_i, [_vp, _i, _u64, _vp, _vp, _i, _sz, _vp, _vp]),
    "shmemg_ibput_on_stream": (_i, [_vp, _u64, _u64, _u64, _u64, _sz, _sz, _i, _i, _vp]),
    "shmemg_ibget_on_stream": (_i, [_vp, _u64, _u64, _u64, _u64, _sz, _sz, _i, _i, _vp]),
    "shmemg_signal_test_on_stream": (_i, [_vp, _u64, _i, _u64, _i, _vp, _vp]),
    "shmemg_signal_test_vec_on_stream": (_i, [_vp, _u64, _sz, _i, _u64, _i, _vp, _vp, _vp]),
    "shmemg_signal_wait_until_all_on_stream": (_i, [_vp, _u64, _sz, _i, _u64, _i, _vp]),
    "shmemg_signal_wait_until_some_on_stream": (_i, [_vp, _u64, _sz, _i, _u64, _i, _vp, _vp, _vp]),
    "shmemg_fcollect_on_stream": (_i, [_vp, _u64, _u64, _sz, _vp]),
    "shmemg_team_split_strided": (_i, [_vp, _i, _i, _i, _i, C.POINTER(_i)]),
    "shmemg_team_n_pes": (_i, [_vp, _i]),
    "shmemg_team_translate_pe": (_i, [_vp, _i, _i]),
    "shmemg_team_reduce_on_stream": (_i, [_vp, _i, _i, _i, _u64, _u64, _sz, _vp]),
    "shmemg_team_fcollect_on_stream": (_i, [_vp, _i, _u64, _u64, _sz, _vp]),
    "shmemg_team_alltoall_on_stream": (_i, [_vp, _i, _u64, _u64, _sz, _vp]),
    "shmemg_team_broadcast_on_stream": (_i, [_vp, _i, _u64, _u64, _sz, _i, _vp]),
    "shmemg_alltoalls_on_stream": (_i, [_vp, _u64, _u64, _u64, _u64, _u64, _u64, _sz, _sz, _vp]),
    "shmemg_cpu_heap_attach": (_i, [_vp, _vp, _sz, _sz]),
    "shmemg_cpu_malloc": (_i, [_vp, _sz, C.POINTER(_u64)]),
    "shmemg_cpu_free": (_i, [_vp, _u64]),
    "shmemg_cpu_ptr": (_vp, [_vp, _u64, _i]),
    "shmemg_put_space_on_stream": (_i, [_vp, _i, _u64, _i, _u64, _sz, _i, _i, _vp]),
    "shmemg_get_space_on_stream": (_i, [_vp, _i, _u64, _i, _u64, _sz, _i, _i, _vp]),
    "shmemg_alltoall_on_stream": (_i, [_vp, _u64, _u64, _sz, _vp]),
    "shmemg_barrier_all_on_stream": (_i, [_vp, _vp]),
    "shmemg_barrier_all_repeat_on_stream": (_i, [_vp, _u32, _u64, _vp]),
    "shmemg_barrier_epoch": (_u64, [_vp, _vp]),
    "shmemg_realign_counters_on_stream": (_i, [_vp, _vp]),
    "shmemg_device_world_get": (_i, [_vp, _vp]),
    "shmemg_ctx_bytes": (_sz, [_u32]),
    "shmemg_ctx_create": (_i, [_vp, _i, _u32, _vp, _sz, _vp, _vp]),
    "shmemg_ctx_counters": (_i, [_vp, _vp, _vp, C.POINTER(_u64), C.POINTER(_u64)]),
    "shmemg_device_exec_ops_ctx_on_stream": (_i, [_vp, _vp, _sz, _vp, _vp, _i, _u32, _vp, C.POINTER(_sz)]),
    "shmemg_put_nbi_on_stream": (_i, [_vp, _u64, _u64, _sz, _i, _i, _vp]),
    "shmemg_get_nbi_on_stream": (_i, [_vp, _u64, _u64, _sz, _i, _i, _vp]),
    "shmemg_put_signal_nbi_on_stream": (_i, [_vp, _u64, _u64, _sz, _u64, _u64, _i, _i, _i, _vp]),
    "shmemg_device_collective_on_stream": (_i, [_vp, _i, _i, _u64, _u64, _sz, _i, _vp]),
    "shmemg_device_exec_ops_on_stream": (_i, [_vp, _vp, _sz, _vp, _vp, C.POINTER(_sz)]),
    "shmemg_app_halo_perturb_on_stream": (_i, [_vp, _u64, _u32, _u64, _u64, _vp]),
    "shmemg_app_halo_pack_on_stream": (_i, [_vp, _u64, _u64, _u32, _vp]),
    "shmemg_app_checksum64_on_stream": (_i, [_vp, _vp, _u64, _u64, _u32, _vp]),
    "shmemg_app_halo_persistent_on_stream": (_i, [_vp, _u64, _u64, _u64, _u32, _u64, _u64, _u32, _vp]),
    "shmemg_probe_atomic_on_stream": (_i, [_vp, _i, _u64, _u64, _sz, _vp]),
    "shmemg_probe_atomic_stream_on_stream": (_i, [_vp, _i, _u64, _vp, _vp, _sz, _i, _vp]),
    "shmemg_probe_copy_all_on_stream": (_i, [_vp, _u64, _u64, _sz, _vp]),
}

_lib = None


def lib():
    """Load libshmemg.so.  Fails loudly: there is no fallback path."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError("libshmemg.so is not built (run `python -c 'import __graft_entry__ as g; g.build()'`); "
                              "the CUDA extension is required, there is no CPU fallback")
        L = C.CDLL(LIB_PATH)
        for name, (res, args) in SYMBOLS.items():
            fn = getattr(L, name)          # AttributeError if the library does not export a declared symbol
            fn.restype, fn.argtypes = res, args
        _lib = L
    return _lib


def _stream(stream=None) -> int:
    s = torch.cuda.current_stream() if stream is None else stream
    return s.cuda_stream


def _dptr(t) -> int:
    if t is None:
        return 0
    assert t.is_cuda and t.is_contiguous()
    return t.data_ptr()


class Batch:
    """A planned op batch (shmemg_batch_t) plus the device plan buffer it lives in."""

    def __init__(self, world: "World", ops: np.ndarray, stream=None):
        assert ops.dtype == OP_DTYPE
        ops = np.ascontiguousarray(ops)
        self.world, self.nops = world, len(ops)
        L = lib()
        nbytes = L.shmemg_batch_plan_bytes(world.h, ops.ctypes.data, len(ops))
        if nbytes == 0:
            raise ShmemgError(ERR.ARG, "shmemg_batch_plan_bytes")
        self.plan = torch.empty(nbytes, dtype=torch.uint8, device=world.device)
        h, bad = C.c_void_p(), C.c_size_t(0)
        rc = L.shmemg_batch_create(world.h, ops.ctypes.data, len(ops), self.plan.data_ptr(), nbytes, _stream(stream),
                                   C.byref(h), C.byref(bad))
        if rc:
            raise ShmemgError(rc, "shmemg_batch_create", "op %d" % bad.value)
        self.h = h
        self.launches = L.shmemg_batch_launches(h)

    def enqueue(self, stream=None):
        self.world._chk(lib().shmemg_batch_enqueue_on_stream(self.world.h, self.h, _stream(stream)),
                        "shmemg_batch_enqueue_on_stream")

    def __del__(self):
        if getattr(self, "h", None) and _lib is not None:
            _lib.shmemg_batch_destroy(self.h)
            self.h = None


class World:
    """npes logical PEs over one device slab (a torch uint8 tensor owned by this object)."""

    def __init__(self, npes: int, heap_bytes: int, device="cuda:0"):
        L = lib()
        if not torch.cuda.is_available():
            raise RuntimeError("no CUDA device: the shmemg hot path has no CPU fallback")
        self.device = torch.device(device)
        need = L.shmemg_slab_bytes_required(npes, heap_bytes)
        if need == 0:
            raise ShmemgError(ERR.ARG, "shmemg_slab_bytes_required")
        self.slab = torch.empty(need, dtype=torch.uint8, device=self.device)   # torch allocations are >= 512-B aligned
        h = C.c_void_p()
        rc = L.shmemg_init(npes, heap_bytes, self.slab.data_ptr(), need, C.byref(h))
        if rc:
            raise ShmemgError(rc, "shmemg_init")
        self.h = h
        self.npes = L.shmemg_n_pes(h)
        self.heap_bytes = L.shmemg_heap_bytes(h)
        self.stride = L.shmemg_heap_stride(h)
        self.launches = 0                  # kernels launched through this object (launch accounting)

    def _chk(self, rc: int, what: str):
        if rc:
            detail = lib().shmemg_last_cuda_error(self.h).decode() if rc == ERR.CUDA else ""
            raise ShmemgError(rc, what, detail)

    def finalize(self):
        if self.h:
            lib().shmemg_finalize(self.h)
            self.h = None

    # ---- capability / allocation / translation -----------------------------------------------------------
    def query_capabilities(self, team: int = TEAM.WORLD) -> int:
        caps = C.c_uint64(0)
        self._chk(lib().shmem_query_capabilities(self.h, team, C.byref(caps)), "shmem_query_capabilities")
        return caps.value

    def malloc(self, nbytes: int) -> int:
        off = C.c_uint64(0)
        self._chk(lib().shmemg_malloc(self.h, nbytes, C.byref(off)), "shmemg_malloc")
        return off.value

    def calloc(self, count: int, size: int, stream=None) -> int:
        off = C.c_uint64(0)
        self._chk(lib().shmemg_calloc(self.h, count, size, C.byref(off), _stream(stream)), "shmemg_calloc")
        return off.value

    def align(self, alignment: int, nbytes: int) -> int:
        off = C.c_uint64(0)
        self._chk(lib().shmemg_align(self.h, alignment, nbytes, C.byref(off)), "shmemg_align")
        return off.value

    def free(self, off: int):
        self._chk(lib().shmemg_free(self.h, off), "shmemg_free")

    def ptr(self, off: int, pe: int) -> int:
        return lib().shmemg_ptr(self.h, off, pe) or 0

    def view(self, off: int, nbytes: int, dtype=torch.uint8) -> torch.Tensor:
        """[npes, nbytes/itemsize] strided torch view of a symmetric object (plumbing: fill / read back)."""
        t = self.slab[: self.npes * self.stride].view(self.npes, self.stride)[:, off:off + nbytes]
        return t if dtype == torch.uint8 else t.view(dtype)

    def heap_write(self, pe: int, dst_off: int, src_host: torch.Tensor, stream=None):
        assert not src_host.is_cuda and src_host.is_contiguous()
        self._chk(lib().shmemg_heap_write_on_stream(self.h, pe, dst_off, src_host.data_ptr(),
                                                    src_host.numel() * src_host.element_size(), _stream(stream)),
                  "shmemg_heap_write_on_stream")

    def heap_read(self, pe: int, dst_host: torch.Tensor, src_off: int, stream=None):
        assert not dst_host.is_cuda and dst_host.is_contiguous()
        self._chk(lib().shmemg_heap_read_on_stream(self.h, pe, dst_host.data_ptr(), src_off,
                                                   dst_host.numel() * dst_host.element_size(), _stream(stream)),
                  "shmemg_heap_read_on_stream")

    # ---- batches and single ops ---------------------------------------------------------------------------------
    def batch(self, ops: np.ndarray, stream=None) -> Batch:
        return Batch(self, ops, stream)

    def enqueue_batch(self, batch: Batch, stream=None):
        batch.enqueue(stream)
        self.launches += batch.launches

    def batch_work_bytes(self, nops: int, payload_bytes: int) -> int:
        return lib().shmemg_batch_work_bytes(self.h, nops, payload_bytes)

    def enqueue_batch_dev(self, ops_dev: torch.Tensor, nops: int, work: torch.Tensor = None, stream=None):
        """One-call form: `ops_dev` is a DEVICE uint8 tensor holding nops shmemg_op_t records; planned on the device.
        work = None uses the world's plan arena (shmemg_enqueue_batch), else shmemg_enqueue_batch_ws."""
        assert ops_dev.is_cuda and ops_dev.is_contiguous() and ops_dev.numel() * ops_dev.element_size() >= nops * 64
        if work is None:
            rc = lib().shmemg_enqueue_batch(self.h, ops_dev.data_ptr(), nops, _stream(stream))
        else:
            rc = lib().shmemg_enqueue_batch_ws(self.h, ops_dev.data_ptr(), nops, work.data_ptr(),
                                               work.numel() * work.element_size(), _stream(stream))
        self._chk(rc, "shmemg_enqueue_batch")
        self.launches += 2 if nops else 0

    def batch_status(self, work: torch.Tensor = None, stream=None):
        """(status, bad_index) of the last one-call batch planned in `work` (None = the arena); synchronises the stream."""
        st, bad = C.c_int(0), C.c_size_t(0)
        self._chk(lib().shmemg_batch_status(self.h, 0 if work is None else work.data_ptr(), _stream(stream), C.byref(st),
                                            C.byref(bad)), "shmemg_batch_status")
        return st.value, bad.value

    def put(self, dest_off, source_off, nbytes, pe, target_pe, stream=None):
        self._chk(lib().shmemg_put_on_stream(self.h, dest_off, source_off, nbytes, pe, target_pe, _stream(stream)),
                  "shmemg_put_on_stream")
        self.launches += 1 if nbytes else 0

    def get(self, dest_off, source_off, nbytes, pe, target_pe, stream=None):
        self._chk(lib().shmemg_get_on_stream(self.h, dest_off, source_off, nbytes, pe, target_pe, _stream(stream)),
                  "shmemg_get_on_stream")
        self.launches += 1 if nbytes else 0

    def put_signal(self, dest_off, source_off, nbytes, sig_off, signal, sig_op, pe, target_pe, stream=None):
        self._chk(lib().shmemg_put_signal_on_stream(self.h, dest_off, source_off, nbytes, sig_off, signal, sig_op, pe,
                                                    target_pe, _stream(stream)), "shmemg_put_signal_on_stream")
        self.launches += 1

    def signal_wait_until(self, sig_off, cmp, value, pe, stream=None):
        self._chk(lib().shmemg_signal_wait_until_on_stream(self.h, sig_off, cmp, value, pe, _stream(stream)),
                  "shmemg_signal_wait_until_on_stream")
        self.launches += 1

    def fence(self, pe, stream=None):
        self._chk(lib().shmemg_fence_on_stream(self.h, pe, _stream(stream)), "shmemg_fence_on_stream")

    def quiet_on_stream(self, pe, stream=None):
        self._chk(lib().shmemg_quiet_on_stream(self.h, pe, _stream(stream)), "shmemg_quiet_on_stream")

    def quiet(self, pe, stream=None):
        self._chk(lib().shmemg_quiet(self.h, pe, _stream(stream)), "shmemg_quiet")

    # ---- device-initiated path (include/shmemg_device.cuh) ---------------------------------------------------------
    def device_exec_ops(self, ops: np.ndarray, stream=None):
        """Run an op list device-initiated: one PE-agent thread block per PE (shmemg_device_exec_ops_on_stream)."""
        assert ops.dtype == OP_DTYPE
        ops = np.ascontiguousarray(ops)
        ops_dev = torch.empty(max(len(ops), 1) * OP_DTYPE.itemsize, dtype=torch.uint8, device=self.device)
        bad = C.c_size_t(0)
        rc = lib().shmemg_device_exec_ops_on_stream(self.h, ops.ctypes.data, len(ops), ops_dev.data_ptr(), _stream(stream),
                                                    C.byref(bad))
        if rc:
            raise ShmemgError(rc, "shmemg_device_exec_ops_on_stream", "op %d" % bad.value)
        self._keep = getattr(self, "_keep", [])
        self._keep.append(ops_dev)                 # must stay valid until the stream has passed the call
        self.launches += 1 if len(ops) else 0

    # ---- explicit device contexts (shmemg_ctx_create; include/shmemg_device.cuh `_nbi` / `shmemg_dev_ctx_*`) -------------
    CTX_DTYPE = np.dtype([("queue", "u8"), ("counters", "u8"), ("capacity", "u4"), ("pe", "i4")])     # shmemg_device_ctx_t

    def ctx_create_all(self, nctx: int, queue_entries: int = 64, stream=None):
        """One context per (PE, c < nctx): returns (host array of handles [npes * nctx], the same array on the device);
        the context memory is a torch tensor kept alive by this object."""
        L = lib()
        per = L.shmemg_ctx_bytes(queue_entries)
        per = (per + 255) // 256 * 256
        mem = torch.empty(self.npes * nctx * per, dtype=torch.uint8, device=self.device)
        handles = np.zeros(self.npes * nctx, dtype=self.CTX_DTYPE)
        for p in range(self.npes):
            for c in range(nctx):
                k = p * nctx + c
                self._chk(L.shmemg_ctx_create(self.h, p, queue_entries, mem.data_ptr() + k * per, per, _stream(stream),
                                              handles[k:k + 1].ctypes.data), "shmemg_ctx_create")
        dev = torch.from_numpy(handles.view(np.uint8).reshape(-1).copy()).to(self.device)
        self._keep = getattr(self, "_keep", []) + [mem, dev]
        return handles, dev

    def ctx_counters(self, handles: np.ndarray, k: int, stream=None):
        a, b = C.c_uint64(0), C.c_uint64(0)
        self._chk(lib().shmemg_ctx_counters(self.h, handles[k:k + 1].ctypes.data, _stream(stream), C.byref(a), C.byref(b)),
                  "shmemg_ctx_counters")
        return a.value, b.value

    def device_exec_ops_ctx(self, ops: np.ndarray, ctxs_dev: torch.Tensor, nctx: int, flags: int = 0, stream=None):
        assert ops.dtype == OP_DTYPE
        ops = np.ascontiguousarray(ops)
        ops_dev = torch.empty(max(len(ops), 1) * OP_DTYPE.itemsize, dtype=torch.uint8, device=self.device)
        bad = C.c_size_t(0)
        rc = lib().shmemg_device_exec_ops_ctx_on_stream(self.h, ops.ctypes.data, len(ops), ops_dev.data_ptr(), ctxs_dev.data_ptr(),
                                                        nctx, flags, _stream(stream), C.byref(bad))
        if rc:
            raise ShmemgError(rc, "shmemg_device_exec_ops_ctx_on_stream", "op %d" % bad.value)
        self._keep = getattr(self, "_keep", []) + [ops_dev]
        self.launches += 1 if len(ops) else 0

    def put_nbi(self, dest_off, source_off, nbytes, pe, target_pe, stream=None):
        self._chk(lib().shmemg_put_nbi_on_stream(self.h, dest_off, source_off, nbytes, pe, target_pe, _stream(stream)),
                  "shmemg_put_nbi_on_stream")
        self.launches += 1 if nbytes else 0

    def get_nbi(self, dest_off, source_off, nbytes, pe, target_pe, stream=None):
        self._chk(lib().shmemg_get_nbi_on_stream(self.h, dest_off, source_off, nbytes, pe, target_pe, _stream(stream)),
                  "shmemg_get_nbi_on_stream")
        self.launches += 1 if nbytes else 0

    def put_signal_nbi(self, dest_off, source_off, nbytes, sig_off, signal, sig_op, pe, target_pe, stream=None):
        self._chk(lib().shmemg_put_signal_nbi_on_stream(self.h, dest_off, source_off, nbytes, sig_off, signal, sig_op, pe,
                                                        target_pe, _stream(stream)), "shmemg_put_signal_nbi_on_stream")
        self.launches += 1

    def device_collective(self, kind, dest_off, source_off, n, dtype=0, root=0, stream=None):
        """One device collective run device-initiated: block p calls shmemg_dev_<kind>_block (include/shmemg_device.cuh)."""
        self._chk(lib().shmemg_device_collective_on_stream(self.h, kind, dtype, dest_off, source_off, n, root, _stream(stream)),
                  "shmemg_device_collective_on_stream")
        self.launches += 1 if n else 0

    def set_dependent_launch(self, enable: bool):
        """Programmatic dependent launch of the executor / planner kernels (on by default; off = plain stream-ordered launches)."""
        self._chk(lib().shmemg_set_dependent_launch(self.h, 1 if enable else 0), "shmemg_set_dependent_launch")

    # ---- SoA AMO batches -------------------------------------------------------------------------------------------
    def set_scratch_for(self, n: int):
        """Register a caller-owned scratch buffer large enough for SHMEMG_AMO_HOT_AGGREGATE calls of up to n ops."""
        need = lib().shmemg_amo_scratch_bytes(self.h, n)
        self._scratch = torch.empty(need, dtype=torch.uint8, device=self.device)
        self._chk(lib().shmemg_set_scratch(self.h, self._scratch.data_ptr(), need), "shmemg_set_scratch")

    def amo_last_path(self) -> int:
        """1 if the last add / fetch-add batch call ran the hot-set kernels, 0 if the plain kernel."""
        return lib().shmemg_amo_last_path(self.h)

    def _hot(self, flags, val, n):
        return bool(flags & AMO_HOT_AGGREGATE) and val is None and n >= (1 << 20) and getattr(self, "_scratch", None) is not None \
            and self._scratch.numel() >= lib().shmemg_amo_scratch_bytes(self.h, n)

    @staticmethod
    def _idx_bytes(elem_idx):
        assert elem_idx.dtype in (torch.int32, torch.int64, torch.uint32, torch.uint64)
        return elem_idx.element_size()

    def atomic_add_batch(self, sym_off, tgt_pe, elem_idx, val=None, val_scalar=0, flags=0, stream=None):
        n = tgt_pe.numel()
        self._chk(lib().shmemg_atomic_add_batch_on_stream(self.h, sym_off, _dptr(tgt_pe), _dptr(elem_idx),
                                                          self._idx_bytes(elem_idx), _dptr(val), val_scalar & NO_STAMP,
                                                          n, flags, _stream(stream)),
                  "shmemg_atomic_add_batch_on_stream")
        self.launches += (2 if self._hot(flags, val, n) else 1) if n or (flags & AMO_THEN_BARRIER) else 0

    def atomic_fetch_add_batch(self, sym_off, tgt_pe, elem_idx, fetched_out, val=None, val_scalar=0, flags=0,
                               stream=None):
        n = tgt_pe.numel()
        self._chk(lib().shmemg_atomic_fetch_add_batch_on_stream(self.h, sym_off, _dptr(tgt_pe), _dptr(elem_idx),
                                                                self._idx_bytes(elem_idx), _dptr(val),
                                                                val_scalar & NO_STAMP, _dptr(fetched_out), n, flags,
                                                                _stream(stream)),
                  "shmemg_atomic_fetch_add_batch_on_stream")
        # launch accounting: SHMEMG_AMO_HOT_AGGREGATE runs a sampling kernel in front of the main one (n >= 2^20, scalar value)
        self.launches += (2 if self._hot(flags, val, n) else 1) if n or (flags & AMO_THEN_BARRIER) else 0

    def atomic_fetch_add_batch_static(self, sym_off, tgt_pe, elem_idx, fetched_out, val_scalar=1, flags=0, stream=None) -> int:
        """Fetch-add with one scalar value for a caller that has no device allocator to draw scratch from (a plug-in given only
        its input / output pointers, a process whose GPU memory is all committed to a pool, a pipeline that cannot afford
        cudaMalloc's device-wide synchronisation): the scratch is a fixed array inside the library, nothing is allocated.  At most
        STATIC_MAX_OPS ops per call (ShmemgError NOMEM with the reason beyond that); calls on one GPU must not overlap, they
        share the array.  Returns 1 when the hot-set kernels ran on the built-in scratch, 0 when the plain kernel ran."""
        n = tgt_pe.numel()
        path = C.c_int(0)
        rc = lib().shmemg_atomic_fetch_add_batch_static_on_stream(self.h, sym_off, _dptr(tgt_pe), _dptr(elem_idx),
                                                                  self._idx_bytes(elem_idx), val_scalar & NO_STAMP,
                                                                  _dptr(fetched_out), n, flags, _stream(stream), C.byref(path))
        if rc:
            raise ShmemgError(rc, "shmemg_atomic_fetch_add_batch_static_on_stream", lib().shmemg_last_cuda_error(self.h).decode())
        self.launches += (1 + path.value) if n or (flags & AMO_THEN_BARRIER) else 0
        return path.value

    def atomic_compare_swap_batch(self, sym_off, tgt_pe, elem_idx, fetched_out, cond=None, cond_scalar=0, val=None,
                                  val_scalar=0, flags=0, stream=None):
        n = tgt_pe.numel()
        self._chk(lib().shmemg_atomic_compare_swap_batch_on_stream(self.h, sym_off, _dptr(tgt_pe), _dptr(elem_idx),
                                                                   self._idx_bytes(elem_idx), _dptr(cond),
                                                                   cond_scalar & NO_STAMP, _dptr(val),
                                                                   val_scalar & NO_STAMP, _dptr(fetched_out), n, flags,
                                                                   _stream(stream)),
                  "shmemg_atomic_compare_swap_batch_on_stream")
        self.launches += 1 if n else 0

    # ---- collectives -------------------------------------------------------------------------------------------------
    def sum_reduce(self, dtype, dest_off, source_off, nreduce, stream=None):
        self._chk(lib().shmemg_sum_reduce_on_stream(self.h, dtype, dest_off, source_off, nreduce, _stream(stream)),
                  "shmemg_sum_reduce_on_stream")
        self.launches += 1 if nreduce else 0

    def reduce(self, op, dtype, dest_off, source_off, nreduce, stream=None):
        self._chk(lib().shmemg_reduce_on_stream(self.h, op, dtype, dest_off, source_off, nreduce, _stream(stream)),
                  "shmemg_reduce_on_stream")
        self.launches += 1 if nreduce else 0

    def broadcast(self, dest_off, source_off, nbytes, root_pe, stream=None):
        self._chk(lib().shmemg_broadcast_on_stream(self.h, dest_off, source_off, nbytes, root_pe, _stream(stream)),
                  "shmemg_broadcast_on_stream")
        self.launches += 1 if nbytes else 0

    def atomic_op_batch(self, amo, width, sym_off, tgt_pe, elem_idx, val=None, val_scalar=0, fetched_out=None, stream=None):
        n = tgt_pe.numel()
        assert elem_idx.numel() == n and (val is None or val.numel() == n) and (fetched_out is None or fetched_out.numel() == n)
        self._chk(lib().shmemg_atomic_op_batch_on_stream(self.h, amo, width, sym_off, _dptr(tgt_pe), _dptr(elem_idx),
                                                         self._idx_bytes(elem_idx), _dptr(val), val_scalar & ((1 << 64) - 1),
                                                         _dptr(fetched_out), n, _stream(stream)),
                  "shmemg_atomic_op_batch_on_stream")
        self.launches += 1 if n else 0

    def atomic_cswap_op_batch(self, width, sym_off, tgt_pe, elem_idx, fetched_out, cond=None, cond_scalar=0, val=None, val_scalar=0,
                              stream=None):
        n = tgt_pe.numel()
        assert elem_idx.numel() == n and (cond is None or cond.numel() == n) and (val is None or val.numel() == n)
        self._chk(lib().shmemg_atomic_cswap_op_batch_on_stream(self.h, width, sym_off, _dptr(tgt_pe), _dptr(elem_idx),
                                                               self._idx_bytes(elem_idx), _dptr(cond), cond_scalar & NO_STAMP,
                                                               _dptr(val), val_scalar & NO_STAMP, _dptr(fetched_out), n,
                                                               _stream(stream)), "shmemg_atomic_cswap_op_batch_on_stream")
        self.launches += 1 if n else 0

    def amo_check_batch(self, width, sym_off, tgt_pe, elem_idx, stream=None):
        """Device-side bounds check of the index arrays of an SoA AMO call: index of the first out-of-range op, or None."""
        out = torch.empty(1, dtype=torch.int64, device=self.device)
        self._chk(lib().shmemg_amo_check_batch_on_stream(self.h, width, sym_off, _dptr(tgt_pe), _dptr(elem_idx),
                                                         self._idx_bytes(elem_idx), tgt_pe.numel(), out.data_ptr(),
                                                         _stream(stream)), "shmemg_amo_check_batch_on_stream")
        self.launches += 1 if tgt_pe.numel() else 0
        v = int(out.item())
        return None if v == -1 else v

    def ibput(self, dest_off, source_off, dst_stride, src_stride, block_bytes, nblocks, pe, target_pe, stream=None):
        self._chk(lib().shmemg_ibput_on_stream(self.h, dest_off, source_off, dst_stride, src_stride, block_bytes, nblocks,
                                               pe, target_pe, _stream(stream)), "shmemg_ibput_on_stream")
        self.launches += 1 if block_bytes and nblocks else 0

    def ibget(self, dest_off, source_off, dst_stride, src_stride, block_bytes, nblocks, pe, target_pe, stream=None):
        self._chk(lib().shmemg_ibget_on_stream(self.h, dest_off, source_off, dst_stride, src_stride, block_bytes, nblocks,
                                               pe, target_pe, _stream(stream)), "shmemg_ibget_on_stream")
        self.launches += 1 if block_bytes and nblocks else 0

    def signal_test(self, sig_off, cmp, value, pe, result_dev, stream=None):
        """result_dev: a 1-element int32 CUDA tensor; read it after synchronising the stream."""
        assert result_dev.dtype == torch.int32
        self._chk(lib().shmemg_signal_test_on_stream(self.h, sig_off, cmp, value & ((1 << 64) - 1), pe, _dptr(result_dev),
                                                     _stream(stream)), "shmemg_signal_test_on_stream")
        self.launches += 1

    # ---- teams (NEXT-3) ---------------------------------------------------------------------------------------------------
    def team_split_strided(self, parent_team, start, stride, size) -> int:
        t = C.c_int(-1)
        self._chk(lib().shmemg_team_split_strided(self.h, parent_team, start, stride, size, C.byref(t)), "shmemg_team_split_strided")
        return t.value

    def team_n_pes(self, team) -> int:
        return lib().shmemg_team_n_pes(self.h, team)

    def team_translate_pe(self, team, rank) -> int:
        return lib().shmemg_team_translate_pe(self.h, team, rank)

    def team_reduce(self, team, op, dtype, dest_off, source_off, nreduce, stream=None):
        self._chk(lib().shmemg_team_reduce_on_stream(self.h, team, op, dtype, dest_off, source_off, nreduce, _stream(stream)),
                  "shmemg_team_reduce_on_stream")
        self.launches += 1 if nreduce else 0

    def team_fcollect(self, team, dest_off, source_off, nbytes, stream=None):
        self._chk(lib().shmemg_team_fcollect_on_stream(self.h, team, dest_off, source_off, nbytes, _stream(stream)),
                  "shmemg_team_fcollect_on_stream")
        self.launches += 1 if nbytes else 0

    def team_alltoall(self, team, dest_off, source_off, nbytes, stream=None):
        self._chk(lib().shmemg_team_alltoall_on_stream(self.h, team, dest_off, source_off, nbytes, _stream(stream)),
                  "shmemg_team_alltoall_on_stream")
        self.launches += 1 if nbytes else 0

    def team_broadcast(self, team, dest_off, source_off, nbytes, root_rank, stream=None):
        self._chk(lib().shmemg_team_broadcast_on_stream(self.h, team, dest_off, source_off, nbytes, root_rank, _stream(stream)),
                  "shmemg_team_broadcast_on_stream")
        self.launches += 1 if nbytes else 0

    def signal_test_vec(self, sig_off, nelems, cmp, value, pe, indices_dev=None, count_dev=None, stream=None):
        self._chk(lib().shmemg_signal_test_vec_on_stream(self.h, sig_off, nelems, cmp, value & ((1 << 64) - 1), pe,
                                                         _dptr(indices_dev), _dptr(count_dev), _stream(stream)),
                  "shmemg_signal_test_vec_on_stream")
        self.launches += 1

    def signal_wait_until_all(self, sig_off, nelems, cmp, value, pe, stream=None):
        self._chk(lib().shmemg_signal_wait_until_all_on_stream(self.h, sig_off, nelems, cmp, value & ((1 << 64) - 1), pe,
                                                               _stream(stream)), "shmemg_signal_wait_until_all_on_stream")
        self.launches += 1

    def signal_wait_until_some(self, sig_off, nelems, cmp, value, pe, indices_dev=None, count_dev=None, stream=None):
        self._chk(lib().shmemg_signal_wait_until_some_on_stream(self.h, sig_off, nelems, cmp, value & ((1 << 64) - 1), pe,
                                                                _dptr(indices_dev), _dptr(count_dev), _stream(stream)),
                  "shmemg_signal_wait_until_some_on_stream")
        self.launches += 1

    def fcollect(self, dest_off, source_off, nbytes, stream=None):
        self._chk(lib().shmemg_fcollect_on_stream(self.h, dest_off, source_off, nbytes, _stream(stream)),
                  "shmemg_fcollect_on_stream")
        self.launches += 1 if nbytes else 0

    def alltoalls(self, dest_off, source_off, dst_pe_stride, src_pe_stride, dst_block_stride, src_block_stride, block_bytes,
                  nblocks, stream=None):
        self._chk(lib().shmemg_alltoalls_on_stream(self.h, dest_off, source_off, dst_pe_stride, src_pe_stride, dst_block_stride,
                                                   src_block_stride, block_bytes, nblocks, _stream(stream)),
                  "shmemg_alltoalls_on_stream")
        self.launches += 1 if block_bytes and nblocks else 0

    # ---- the CPU space of the two-space model ------------------------------------------------------------------------------
    def cpu_heap_attach(self, heap_bytes: int):
        """Attach a CPU space of heap_bytes per PE in pinned host memory owned by this object."""
        stride = (heap_bytes + 511) // 512 * 512
        self.cpu_slab = torch.empty(self.npes * stride, dtype=torch.uint8).pin_memory()
        self.cpu_stride = stride
        self._chk(lib().shmemg_cpu_heap_attach(self.h, self.cpu_slab.data_ptr(), heap_bytes, self.cpu_slab.numel()),
                  "shmemg_cpu_heap_attach")

    def cpu_malloc(self, nbytes: int) -> int:
        off = C.c_uint64(0)
        self._chk(lib().shmemg_cpu_malloc(self.h, nbytes, C.byref(off)), "shmemg_cpu_malloc")
        return off.value

    def cpu_free(self, off: int):
        self._chk(lib().shmemg_cpu_free(self.h, off), "shmemg_cpu_free")

    def cpu_ptr(self, off: int, pe: int) -> int:
        return lib().shmemg_cpu_ptr(self.h, off, pe) or 0

    def cpu_view(self, off: int, nbytes: int) -> torch.Tensor:
        """[npes, nbytes] HOST view of an object of the CPU space."""
        return self.cpu_slab.view(self.npes, self.cpu_stride)[:, off:off + nbytes]

    def put_space(self, dst_space, dest_off, src_space, source_off, nbytes, pe, target_pe, stream=None):
        self._chk(lib().shmemg_put_space_on_stream(self.h, dst_space, dest_off, src_space, source_off, nbytes, pe, target_pe,
                                                   _stream(stream)), "shmemg_put_space_on_stream")
        self.launches += 1 if nbytes and dst_space == 0 and src_space == 0 else 0

    def get_space(self, dst_space, dest_off, src_space, source_off, nbytes, pe, target_pe, stream=None):
        self._chk(lib().shmemg_get_space_on_stream(self.h, dst_space, dest_off, src_space, source_off, nbytes, pe, target_pe,
                                                   _stream(stream)), "shmemg_get_space_on_stream")
        self.launches += 1 if nbytes and dst_space == 0 and src_space == 0 else 0

    # ---- PE -> GPU sharding (NEXT-4 (iii)): this world is one shard of a multi-GPU world; g-calls take GLOBAL PE numbers ----
    def shard_init(self, nshards: int, my_shard: int):
        self._chk(lib().shmemg_shard_init(self.h, nshards, my_shard), "shmemg_shard_init")
        self.nshards, self.shard = nshards, my_shard

    def shard_export(self):
        """(64-byte CUDA IPC handle of this world's slab allocation, offset of the slab inside it): carry both to the peers."""
        buf, off = C.create_string_buffer(64), C.c_uint64(0)
        self._chk(lib().shmemg_shard_export(self.h, buf, C.byref(off)), "shmemg_shard_export")
        return bytes(buf.raw), off.value

    def shard_attach_ipc(self, shard: int, handle: bytes, offset: int):
        assert len(handle) == 64
        self._chk(lib().shmemg_shard_attach_ipc(self.h, shard, C.create_string_buffer(handle, 64), offset), "shmemg_shard_attach_ipc")

    def shard_attach_world(self, shard: int, other: "World"):
        """A shard that lives in THIS process (its slab is addressable here: same device, or peer access enabled)."""
        self._chk(lib().shmemg_shard_attach_ptr(self.h, shard, other.slab.data_ptr()), "shmemg_shard_attach_ptr")

    def shard_global_npes(self) -> int:
        return lib().shmemg_shard_global_npes(self.h)

    def gput(self, dest_off, source_off, nbytes, gpe, target_gpe, stream=None):
        self._chk(lib().shmemg_gput_on_stream(self.h, dest_off, source_off, nbytes, gpe, target_gpe, _stream(stream)), "shmemg_gput_on_stream")
        self.launches += 1 if nbytes else 0

    def gget(self, dest_off, source_off, nbytes, gpe, target_gpe, stream=None):
        self._chk(lib().shmemg_gget_on_stream(self.h, dest_off, source_off, nbytes, gpe, target_gpe, _stream(stream)), "shmemg_gget_on_stream")
        self.launches += 1 if nbytes else 0

    def gput_signal(self, dest_off, source_off, nbytes, sig_off, signal, sig_op, gpe, target_gpe, stream=None):
        self._chk(lib().shmemg_gput_signal_on_stream(self.h, dest_off, source_off, nbytes, sig_off, signal & NO_STAMP, sig_op, gpe,
                                                     target_gpe, _stream(stream)), "shmemg_gput_signal_on_stream")
        self.launches += 1

    def gsignal_wait_until(self, sig_off, cmp, value, gpe, stream=None):
        self._chk(lib().shmemg_gsignal_wait_until_on_stream(self.h, sig_off, cmp, value & NO_STAMP, gpe, _stream(stream)),
                  "shmemg_gsignal_wait_until_on_stream")
        self.launches += 1

    def gatomic_batch(self, op, sym_off, target_gpe, elem_idx, val=None, val_scalar=0, cond=None, cond_scalar=0, fetched_out=None,
                      stream=None):
        n = target_gpe.numel()
        self._chk(lib().shmemg_gatomic_batch_on_stream(self.h, op, sym_off, _dptr(target_gpe), _dptr(elem_idx), self._idx_bytes(elem_idx),
                                                       _dptr(cond), cond_scalar & NO_STAMP, _dptr(val), val_scalar & NO_STAMP,
                                                       _dptr(fetched_out), n, _stream(stream)), "shmemg_gatomic_batch_on_stream")
        self.launches += 1 if n else 0

    def galltoall(self, dest_off, source_off, nbytes, stream=None):
        self._chk(lib().shmemg_galltoall_on_stream(self.h, dest_off, source_off, nbytes, _stream(stream)), "shmemg_galltoall_on_stream")
        self.launches += 1 if nbytes else 0

    def gfcollect(self, dest_off, source_off, nbytes, stream=None):
        self._chk(lib().shmemg_gfcollect_on_stream(self.h, dest_off, source_off, nbytes, _stream(stream)), "shmemg_gfcollect_on_stream")
        self.launches += 1 if nbytes else 0

    def gsum_reduce(self, dtype, dest_off, source_off, nreduce, stream=None):
        self._chk(lib().shmemg_gsum_reduce_on_stream(self.h, dtype, dest_off, source_off, nreduce, _stream(stream)),
                  "shmemg_gsum_reduce_on_stream")
        self.launches += 1 if nreduce else 0

    def gbarrier_all(self, stream=None):
        self._chk(lib().shmemg_gbarrier_all_on_stream(self.h, _stream(stream)), "shmemg_gbarrier_all_on_stream")
        self.launches += 1

    def alltoall(self, dest_off, source_off, nbytes, stream=None):
        self._chk(lib().shmemg_alltoall_on_stream(self.h, dest_off, source_off, nbytes, _stream(stream)),
                  "shmemg_alltoall_on_stream")
        self.launches += 1 if nbytes else 0

    def barrier_all(self, stream=None):
        self._chk(lib().shmemg_barrier_all_on_stream(self.h, _stream(stream)), "shmemg_barrier_all_on_stream")
        self.launches += 1

    def barrier_all_repeat(self, count, stamp_off=NO_STAMP, stream=None):
        self._chk(lib().shmemg_barrier_all_repeat_on_stream(self.h, count, stamp_off, _stream(stream)),
                  "shmemg_barrier_all_repeat_on_stream")
        self.launches += 1 if count else 0

    def realign_counters(self, stream=None):
        """After a kernel that did not finish its barrier rounds: round the monotonic arrival counters up to a round boundary."""
        self._chk(lib().shmemg_realign_counters_on_stream(self.h, _stream(stream)), "shmemg_realign_counters_on_stream")
        self.launches += 1

    def barrier_epoch(self, stream=None) -> int:
        return lib().shmemg_barrier_epoch(self.h, _stream(stream))

    # ---- ceiling probes (include/shmemg_probe.h; measurement utilities, not library ops) ------------------------------
    def probe_atomic(self, mode, sym_off, words_per_pe, n, stream=None):
        self._chk(lib().shmemg_probe_atomic_on_stream(self.h, mode, sym_off, words_per_pe, n, _stream(stream)),
                  "shmemg_probe_atomic_on_stream")

    def probe_atomic_stream(self, mode, sym_off, tgt_pe, elem_idx, n, aggregate=False, stream=None):
        self._chk(lib().shmemg_probe_atomic_stream_on_stream(self.h, mode, sym_off, _dptr(tgt_pe), _dptr(elem_idx), n,
                                                             1 if aggregate else 0, _stream(stream)),
                  "shmemg_probe_atomic_stream_on_stream")

    def probe_copy_all(self, dst_off, src_off, nbytes, stream=None):
        self._chk(lib().shmemg_probe_copy_all_on_stream(self.h, dst_off, src_off, nbytes, _stream(stream)),
                  "shmemg_probe_copy_all_on_stream")

    # ---- halo application kernels (include/shmemg_app.h; not library ops) ---------------------------------------------
    def app_halo_perturb(self, U_off, B, seed, rnd, stream=None):
        self._chk(lib().shmemg_app_halo_perturb_on_stream(self.h, U_off, B, seed, rnd, _stream(stream)),
                  "shmemg_app_halo_perturb_on_stream")

    def app_halo_pack(self, send_off, U_off, B, stream=None):
        self._chk(lib().shmemg_app_halo_pack_on_stream(self.h, send_off, U_off, B, _stream(stream)),
                  "shmemg_app_halo_pack_on_stream")

    def app_halo_persistent(self, U_off, ghost_off, sig_off, B, seed, first_round, rounds, stream=None):
        self._chk(lib().shmemg_app_halo_persistent_on_stream(self.h, U_off, ghost_off, sig_off, B, seed, first_round, rounds,
                                                             _stream(stream)), "shmemg_app_halo_persistent_on_stream")

    def app_checksum64(self, out, sym_off, seg_bytes, nseg, stream=None):
        self._chk(lib().shmemg_app_checksum64_on_stream(self.h, _dptr(out), sym_off, seg_bytes, nseg, _stream(stream)),
                  "shmemg_app_checksum64_on_stream")
