"""GPU parity of the sharded world (NEXT-4 (iii): PE -> GPU sharding over a load-store fabric, include/shmemg.h) against the
GLOBAL oracle world.  Only one GPU is available, so the shards are (1) two worlds of ONE process attached by pointer -- every
kernel, the address translation, system-scope AMOs and signals, the stream barrier of the shards on two streams; (2) two
PROCESSES with one world each, their slabs mapped into each other through CUDA IPC (`sharding.connect_shards` over gloo), with
host-level synchronisation between the phases (no kernel of one process ever waits for a kernel of the other)."""
import json
import os
import socket
import subprocess
import sys

import numpy as np
import pytest
import torch

from paper_2607_08006_b200 import ERR, OP, ShmemgError, World
from paper_2607_08006_b200.binding import CAP, TEAM

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, os.path.join(ROOT, "tests"))
import shard_common as sc  # noqa: E402


def _in_process(G, L):
    case = sc.Case(G, L)
    rs = [sc.ShardRunner(case, s) for s in range(G)]
    for s, r in enumerate(rs):
        r.w.shard_init(G, s)
    for s, r in enumerate(rs):
        for t, q in enumerate(rs):
            if t != s:
                r.w.shard_attach_world(t, q.w)
    return case, rs


@pytest.mark.parametrize("G,L", [(2, 3), (3, 2), (1, 4)])
def test_sharded_world_in_one_process_matches_the_global_oracle(G, L):
    case, rs = _in_process(G, L)
    assert rs[0].w.shard_global_npes() == G * L
    for ph in case.phases:
        for r in rs:
            r.run_phase(ph)
        torch.cuda.synchronize()
    for r in rs:
        r.run_amos()
    torch.cuda.synchronize()
    for r in rs:
        r.run_alltoall()
    torch.cuda.synchronize()
    sc.check(case, [r.results() for r in rs])
    caps = rs[0].w.query_capabilities(TEAM.WORLD)
    assert bool(caps & CAP.PEER_SHARDS) == (G > 1)


def test_stream_barrier_of_the_shards_on_two_streams():
    """shmemg_gbarrier_all_on_stream: shard 0 puts into shard 1 on its stream, both enqueue the barrier on their OWN streams,
    shard 1 then reads what arrived.  Without the barrier nothing orders stream 1 after stream 0.  Run in a subprocess with a
    timeout: two kernels that wait for each other need both streams to make progress."""
    code = r"""
import sys
sys.path.insert(0, %r); sys.path.insert(0, %r)
import numpy as np, torch
import shard_common as sc
case = sc.Case(2, 2)
rs = [sc.ShardRunner(case, s) for s in range(2)]
for s, r in enumerate(rs): r.w.shard_init(2, s)
rs[0].w.shard_attach_world(1, rs[1].w); rs[1].w.shard_attach_world(0, rs[0].w)
st = [torch.cuda.Stream(), torch.cuda.Stream()]
n = 20000
spin = torch.empty(1 << 26, dtype=torch.float32, device="cuda:0")
for rnd in range(1, 6):
    with torch.cuda.stream(st[0]):
        spin.add_(1.0)                                             # stream 0 is late
        rs[0].w.view(rs[0].off["src"], n).fill_(rnd)
        rs[0].w.gput(rs[0].off["dst"], rs[0].off["src"], n, 0, 1)  # global PE 0 (shard 0) -> global PE 1 (shard 1, local 0)
        rs[0].w.gbarrier_all()
    with torch.cuda.stream(st[1]):
        rs[1].w.gbarrier_all()
        got = rs[1].w.view(rs[1].off["dst"], n)[0].clone()
    torch.cuda.synchronize()
    assert (got == rnd).all(), rnd
print("BARRIER OK")
""" % (ROOT, os.path.join(ROOT, "tests"))
    p = subprocess.run([sys.executable, "-c", code], capture_output=True, text=True, timeout=300)
    assert p.returncode == 0 and "BARRIER OK" in p.stdout, p.stderr[-2000:]


def test_shard_argument_checks():
    w = World(2, 1 << 16, sc.DEV)
    with pytest.raises(ShmemgError) as e:
        w.gput(0, 256, 16, 0, 1)                      # before shmemg_shard_init
    assert e.value.code == ERR.ARG
    w.shard_init(2, 0)
    with pytest.raises(ShmemgError) as e:
        w.gput(0, 256, 16, 0, 1)                      # shard 1 not attached
    assert e.value.code == ERR.ARG
    w2 = World(2, 1 << 16, sc.DEV)
    w2.shard_init(2, 1)
    from paper_2607_08006_b200.binding import lib
    host = torch.empty(1 << 20, dtype=torch.uint8).pin_memory()
    assert lib().shmemg_shard_attach_ptr(w.h, 1, host.data_ptr()) == ERR.ARG      # a peer slab must be DEVICE memory this GPU can reach
    assert b"not device memory" in lib().shmemg_last_cuda_error(w.h)
    with pytest.raises(ShmemgError) as e:
        w.gput(0, 256, 16, 0, 1)                      # the refused attach left shard 1 unattached
    assert e.value.code == ERR.ARG
    w.shard_attach_world(1, w2)
    with pytest.raises(ShmemgError) as e:
        w.gput(0, 256, 16, 1, 0)                      # global PE 1 lives on shard 1: not a local initiator
    assert e.value.code == ERR.PE
    with pytest.raises(ShmemgError) as e:
        w.gput(0, 256, 16, 0, 4)                      # 4 global PEs: 0 .. 3
    assert e.value.code == ERR.PE
    with pytest.raises(ShmemgError) as e:
        w.gput((1 << 16) - 8, 0, 16, 0, 1)
    assert e.value.code == ERR.RANGE
    with pytest.raises(ShmemgError) as e:
        w.shard_init(2, 0)                            # once
    assert e.value.code == ERR.ARG
    w.gput(0, 256, 0, 0, 3)                           # zero bytes: nothing enqueued
    torch.cuda.synchronize()


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def test_two_processes_over_cuda_ipc_match_the_global_oracle(tmp_path):
    port = _free_port()
    procs = []
    for r in range(2):
        env = dict(os.environ, MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(r), WORLD_SIZE="2")
        procs.append(subprocess.Popen([sys.executable, os.path.join(ROOT, "tests", "shard_worker.py"), str(tmp_path)], env=env,
                                      stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True))
    for p in procs:
        out, err = p.communicate(timeout=600)
        assert p.returncode == 0, err[-3000:]
    case = sc.Case(2, 3)
    results = []
    for r in range(2):
        z = np.load(os.path.join(str(tmp_path), "shard%d.npz" % r))
        results.append({k: z[k] for k in z.files})
    sc.check(case, results)
