"""Load a neutral workload description (an object with npes / obj_names / obj_bytes / init / ops, as built by
workloads.spec.Program) into a World: allocate its objects with shmemg_malloc, upload initial contents and
translate the op records into shmemg_op_t descriptors.  Marshalling only."""
from __future__ import annotations

import numpy as np
import torch

from .binding import OP_DTYPE, World


class Loaded:
    def __init__(self, world: World, prog):
        assert prog.npes == world.npes
        self.world = world
        self.off = {}
        for name, nb in zip(prog.obj_names, prog.obj_bytes):
            off = world.malloc(nb)
            self.off[name] = (off, nb)
            v = world.view(off, nb)
            if name in prog.init:
                v.copy_(torch.from_numpy(np.ascontiguousarray(prog.init[name])))
            else:
                v.zero_()
        self.names = list(prog.obj_names)
        torch.cuda.synchronize()

    def translate(self, prog) -> np.ndarray:
        ops = prog.ops
        base = np.array([self.off[n][0] for n in self.names] + [0], dtype=np.uint64)   # index -1 -> 0
        out = np.zeros(len(ops), dtype=OP_DTYPE)
        out["opcode"] = ops["kind"]            # neutral kinds 1..10 coincide with SHMEMG_OP_* by construction
        out["sig_op"] = ops["sig_op"]
        out["cmp"] = ops["cmp"]
        out["ctx"] = ops["ctx"]
        out["initiator_pe"] = ops["initiator"]
        out["target_pe"] = ops["target"]
        out["rem_off"] = base[ops["rem_obj"]] + ops["rem_off"]
        out["loc_off"] = base[ops["loc_obj"]] + ops["loc_off"]
        out["sig_off"] = base[ops["sig_obj"]] + ops["sig_off"]
        out["nbytes"] = ops["nbytes"]
        out["value"] = ops["value"]
        out["cond"] = ops["cond"]
        return out

    def obj(self, name: str, dtype=torch.uint8) -> torch.Tensor:
        off, nb = self.off[name]
        return self.world.view(off, nb, dtype)

    def obj_numpy(self, name: str, dtype=np.uint8) -> np.ndarray:
        return self.obj(name).cpu().numpy().view(dtype)
