"""One process = one shard (tests/test_gpu_shard.py::test_two_processes_over_cuda_ipc_match_the_global_oracle).
RANK / WORLD_SIZE / MASTER_* from the environment; both shards use cuda:0 (only one GPU exists here), their slabs mapped into each
other through CUDA IPC.  The phases are separated by a HOST barrier (device synchronise + gloo barrier): no kernel of this
process waits for a kernel of the other one."""
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
sys.path.insert(0, os.path.join(ROOT, "tests"))

import numpy as np  # noqa: E402
import torch  # noqa: E402
import torch.distributed as dist  # noqa: E402

import shard_common as sc  # noqa: E402
from paper_2607_08006_b200.sharding import connect_shards  # noqa: E402


def main():
    out_dir = sys.argv[1]
    rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
    dist.init_process_group("gloo", rank=rank, world_size=world)
    torch.cuda.set_device(0)
    case = sc.Case(world, 3)
    r = sc.ShardRunner(case, rank)
    connect_shards(r.w, dist)

    def sync():
        torch.cuda.synchronize()
        dist.barrier()
    sync()
    for ph in case.phases:
        r.run_phase(ph)
        sync()
    r.run_amos()                       # both processes' system-scope atomics hit the same words at the same time
    sync()
    r.run_alltoall()
    sync()
    np.savez(os.path.join(out_dir, "shard%d.npz" % rank), **r.results())
    sync()                             # nobody unmaps a slab the other one may still read
    r.w.finalize()
    dist.destroy_process_group()


if __name__ == "__main__":
    main()
