"""Bootstrap of a sharded world (include/shmemg.h "PE -> GPU sharding"): one process per GPU, `torch.distributed` carries the
CUDA IPC handles of the slabs between the processes -- plumbing only; every data-path step runs in the library's kernels
over the peer mappings.  The process group may use any backend (the handles are host bytes); nothing here is a data-path
collective."""
from __future__ import annotations


def exchange(dist, item):
    """[item of rank 0, item of rank 1, ...] on every rank (an all-gather of small picklable host objects)."""
    out = [None] * dist.get_world_size()
    dist.all_gather_object(out, item)
    return out


def connect_shards(world, dist):
    """Make `world` shard RANK of a WORLD_SIZE-shard world: export this slab, gather everybody's handle, map the peers.
    Every rank must call it (collective), with worlds of the same npes / heap size that have made the same allocations."""
    n, me = dist.get_world_size(), dist.get_rank()
    world.shard_init(n, me)
    geo = (world.npes, world.heap_bytes)
    handles = exchange(dist, (geo,) + tuple(world.shard_export()))
    for r, (g, handle, offset) in enumerate(handles):
        if g != geo:
            raise ValueError("shard %d has geometry %r, this one %r: the shards of one world are symmetric" % (r, g, geo))
        if r != me:
            world.shard_attach_ipc(r, handle, offset)
    dist.barrier()                     # nobody starts issuing before every mapping exists
    return world
