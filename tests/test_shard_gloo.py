"""NEXT-4 (iii), host side, without a GPU: the C-ABI placement functions against the oracle's definition, and the bootstrap of
a sharded world (`paper_2607_08006_b200.sharding.connect_shards`) over gloo with world_size 2 on a stand-in world object --
the handle exchange, the symmetric-geometry check and the attach calls each rank makes."""
import json
import os
import socket
import subprocess
import sys

import pytest

from oracle import oracle as orc
from paper_2607_08006_b200 import binding

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_c_abi_placement_equals_the_oracle_definition():
    L = binding.lib()
    for G in (1, 2, 3, 8, 16):
        for g in range(4 * G + 3):
            assert L.shmemg_shard_of(g, G) == orc.shard_of(g, G)
            assert L.shmemg_shard_local_index(g, G) == orc.shard_local_index(g, G)
            assert L.shmemg_shard_global_pe(orc.shard_of(g, G), orc.shard_local_index(g, G), G) == g
    assert L.shmemg_shard_of(-1, 2) == binding.ERR.ARG and L.shmemg_shard_of(3, 0) == binding.ERR.ARG
    assert L.shmemg_shard_global_pe(2, 0, 2) == binding.ERR.ARG and L.shmemg_shard_local_index(-5, 2) == binding.ERR.ARG


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


_WORKER = r"""
import json, os, sys
sys.path.insert(0, sys.argv[1])
import torch.distributed as dist
from paper_2607_08006_b200.sharding import connect_shards
rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
dist.init_process_group("gloo", rank=rank, world_size=world)
class FakeWorld:                      # records what connect_shards asks of a world (no GPU here)
    def __init__(self, npes, heap):
        self.npes, self.heap_bytes, self.calls = npes, heap, []
    def shard_init(self, n, me): self.calls.append(["init", n, me])
    def shard_export(self): return bytes([rank + 1]) * 64, 4096 * (rank + 1)
    def shard_attach_ipc(self, shard, handle, offset): self.calls.append(["attach", shard, handle[0], len(handle), offset])
w = connect_shards(FakeWorld(4, 1 << 20), dist)
err = ""
try:
    connect_shards(FakeWorld(4 + rank, 1 << 20), dist)       # asymmetric geometry must be refused on every rank
except ValueError as e:
    err = str(e)[:20]
dist.barrier()
dist.destroy_process_group()
print("RESULT " + json.dumps([rank, w.calls, err]))
"""


def test_connect_shards_world_size_2_gloo():
    port = _free_port()
    procs = []
    for r in range(2):
        env = dict(os.environ, MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(r), WORLD_SIZE="2")
        procs.append(subprocess.Popen([sys.executable, "-c", _WORKER, ROOT], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True))
    res = []
    for p in procs:
        out, err = p.communicate(timeout=240)
        assert p.returncode == 0, err[-2000:]
        res.append(json.loads([ln for ln in out.splitlines() if ln.startswith("RESULT ")][0][7:]))
    res.sort()
    # rank 0 declares itself shard 0 of 2 and maps shard 1 with rank 1's handle and offset, and vice versa
    assert res[0][1] == [["init", 2, 0], ["attach", 1, 2, 64, 8192]]
    assert res[1][1] == [["init", 2, 1], ["attach", 0, 1, 64, 4096]]
    assert res[0][2].startswith("shard") and res[1][2].startswith("shard")
