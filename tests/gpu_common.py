"""Helpers shared by the GPU parity tests: run a neutral Program through the CUDA path (C-ABI via the
binding) and through the oracle, and compare object by object."""
from __future__ import annotations

import numpy as np
import torch

from oracle import oracle as orc
from paper_2607_08006_b200 import World
from paper_2607_08006_b200.loader import Loaded

DEV = "cuda:0"


def heap_bytes_for(prog, slack=4096):
    return sum((b + 255) // 256 * 256 for b in prog.obj_bytes) + slack


def run_gpu(prog, batches=None, heap_bytes=None):
    """batches: list of Programs sharing prog's objects (default: [prog]); each is one enqueue."""
    hb = heap_bytes or heap_bytes_for(prog)
    w = World(prog.npes, hb, DEV)
    ld = Loaded(w, prog)
    for q in (batches or [prog]):
        b = w.batch(ld.translate(q))
        w.enqueue_batch(b)
    w.quiet(0)
    return w, ld


def ops_to_dev(ops: np.ndarray) -> torch.Tensor:
    """shmemg_op_t records as a DEVICE uint8 tensor (input of the one-call form shmemg_enqueue_batch)."""
    return torch.from_numpy(np.ascontiguousarray(ops).view(np.uint8).reshape(-1).copy()).to(DEV)


def run_gpu_onecall(prog, batches=None, heap_bytes=None, arena=False):
    """Same as run_gpu, through the ONE-CALL form: the descriptors are device-resident and planned on the device
    (shmemg_enqueue_batch / shmemg_enqueue_batch_ws); the plan status is checked after every batch."""
    hb = heap_bytes or heap_bytes_for(prog)
    w = World(prog.npes, hb, DEV)
    ld = Loaded(w, prog)
    keep = []
    for q in (batches or [prog]):
        ops = ld.translate(q)
        od = ops_to_dev(ops) if len(ops) else torch.zeros(64, dtype=torch.uint8, device=DEV)
        work = None
        if not arena:
            payload = int(ops["nbytes"][(ops["opcode"] >= 1) & (ops["opcode"] <= 3)].sum())
            work = torch.empty(w.batch_work_bytes(len(ops), payload), dtype=torch.uint8, device=DEV)
        w.enqueue_batch_dev(od, len(ops), work)
        if len(ops):
            assert w.batch_status(work) == (0, 0)
        keep.append((od, work))
    w.quiet(0)
    return w, ld


def run_gpu_device(prog, batches=None, heap_bytes=None):
    """Same as run_gpu, but DEVICE-INITIATED: every batch is executed by PE-agent thread blocks through the
    entry points of include/shmemg_device.cuh (shmemg_device_exec_ops_on_stream)."""
    hb = heap_bytes or heap_bytes_for(prog)
    w = World(prog.npes, hb, DEV)
    ld = Loaded(w, prog)
    for q in (batches or [prog]):
        w.device_exec_ops(ld.translate(q))
    w.quiet(0)
    return w, ld


def run_gpu_device_ctx(prog, batches=None, heap_bytes=None, queue_entries=8):
    """DEVICE-INITIATED with EXPLICIT CONTEXTS: one context handle per (PE, context) created on the host and cached in device
    memory; puts / gets / put_signals are non-blocking on their op's context (shmemg_device_exec_ops_ctx_on_stream).  The small
    queue (8 entries) also exercises the drain-when-full path."""
    hb = heap_bytes or heap_bytes_for(prog)
    w = World(prog.npes, hb, DEV)
    ld = Loaded(w, prog)
    nctx = 1
    for q in (batches or [prog]):
        if len(q.ops):
            nctx = max(nctx, int(q.ops["ctx"].max()) + 1)
    handles, dev = w.ctx_create_all(nctx, queue_entries)
    for q in (batches or [prog]):
        w.device_exec_ops_ctx(ld.translate(q), dev, nctx)
    w.quiet(0)
    w._ctx_handles = handles
    return w, ld


def run_oracle(prog, batches=None, heap_bytes=None):
    hb = heap_bytes or heap_bytes_for(prog)
    ow = orc.OracleWorld(prog.npes, hb)
    ow.load_program(prog)
    for q in (batches or [prog]):
        ow.run_program(q)
    return ow


def assert_objects_equal(prog, ld, ow, names=None):
    for name in (names or prog.obj_names):
        g = ld.obj_numpy(name)
        o = ow.obj(name)
        if not np.array_equal(g, o):
            bad = np.argwhere(g != o)
            raise AssertionError("object %r differs at %d bytes; first (pe, byte) = %s" % (name, len(bad), bad[0]))


def to_dev(a: np.ndarray) -> torch.Tensor:
    a = np.ascontiguousarray(a)
    if a.dtype == np.uint64:
        a = a.view(np.int64)
    if a.dtype == np.uint32:
        a = a.view(np.int32)
    return torch.from_numpy(a).to(DEV)
