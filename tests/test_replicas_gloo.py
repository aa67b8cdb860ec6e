"""The N > 1 path of bench.py on CPU: two processes over gloo (world_size 2).  The hot path does not shard (DESIGN.md 9:
replicas only), so what N > 1 adds is the max-over-ranks reduction of the segment times and the whole-job unit count;
both are exercised here without a GPU."""
import os
import socket
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


_WORKER = r"""
import json, os, sys
sys.path.insert(0, sys.argv[1])
import torch
import torch.distributed as dist
import bench
rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
dist.init_process_group("gloo", rank=rank, world_size=world)
seg = {"alltoall": 1.0 + rank, "halo_put_signal_wait": 5.0 - rank, "atomic_add": 0.5}
e2e = {"alltoall": 10.0 * (rank + 1), "halo_put_signal_wait": 7.0, "atomic_add": 3.0 - rank}
names, seg_r, whole_r, e2e_r = bench.max_over_ranks(dist, torch.device("cpu"), seg, 100.0 + rank, e2e)
dist.barrier()
dist.destroy_process_group()
print("RESULT " + json.dumps([rank, names, seg_r, whole_r, e2e_r]))
"""


def test_max_over_ranks_and_whole_job_units_world_size_2():
    import json
    import subprocess
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
    names = res[0][1]
    for rank, names, seg, whole, e2e in res:                       # every rank sees the same reduced values
        assert names == ["alltoall", "atomic_add", "halo_put_signal_wait"]
        assert seg == {"alltoall": 2.0, "atomic_add": 0.5, "halo_put_signal_wait": 5.0}
        assert whole == 101.0
        assert e2e == {"alltoall": 20.0, "atomic_add": 3.0, "halo_put_signal_wait": 7.0}
    sys.path.insert(0, ROOT)
    import bench
    table = {"alltoall": dict(cls="copy", bytes=1000, launches=1), "atomic_add": dict(cls="amo", ops=10, launches=2),
             "halo_put_signal_wait": dict(cls="copy", bytes=500, launches=50)}
    units = bench.whole_job_units(table, names, steps=3, world=2)
    assert units == {"alltoall": 6000, "atomic_add": 60, "halo_put_signal_wait": 3000}
    secs = {k: v * 1e-3 for k, v in res[0][2].items()}
    gbps, mops, cs, as_ = bench.class_rates(table, secs, units)
    assert gbps == pytest.approx(9000 / 7e-3 / 1e9) and mops == pytest.approx(60 / 0.5e-3 / 1e6)


def test_single_process_path_needs_no_process_group():
    sys.path.insert(0, ROOT)
    import torch
    import bench
    names, seg, whole, e2e = bench.max_over_ranks(None, torch.device("cpu"), {"b": 2.0, "a": 1.0}, 3.0, None)
    assert names == ["a", "b"] and seg == {"a": 1.0, "b": 2.0} and whole == 3.0 and e2e is None
