"""Writes tests/golden/oracle_checksums.txt: checksums of what the CPU ORACLE computes on small seeded instances of the five
configurations.  Calls only oracle/ and the seeded input generators (workloads/); nothing here comes from the CUDA path.

The paper prints no numeric example ("This paper focuses on specification design rather than benchmarking"),
so there is no value of the paper's to store; these are regression pins of the oracle against itself over time (a change of
its arithmetic shows up here and must be justified in the commit that regenerates the file).  The pins that check the
oracle against things OTHER than itself are in tests/test_oracle_pins*.py.

    python tests/golden/make_golden.py          # rewrites the file
"""
from __future__ import annotations

import hashlib
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

from oracle import oracle as orc  # noqa: E402
from workloads import configs, gen  # noqa: E402

OUT = os.path.join(os.path.dirname(os.path.abspath(__file__)), "oracle_checksums.txt")


def digest(a: np.ndarray) -> str:
    return hashlib.sha256(np.ascontiguousarray(a).tobytes()).hexdigest()[:32]


def cases():
    # C1 at full size: 65 536 atomic adds on 4 x 16 384 int64 (BASELINE.json configs[0])
    wl = configs.c1_atomic_add()
    w = orc.OracleWorld(wl.npes, wl.nelem * 8 + 4096)
    a = w.malloc(wl.nelem * 8)
    w.atomic_add_batch(a, wl.tgt_pe, wl.idx, wl.val)
    yield "c1_atomic_add_full", digest(w.view(a, wl.nelem * 8))
    # C3a shape, 8 PEs x 4 KiB blocks
    npes, blk = 8, 4096
    w = orc.OracleWorld(npes, 4 * npes * blk)
    s, d = w.malloc(npes * blk), w.malloc(npes * blk)
    w.view(s, npes * blk)[:] = configs.c3a_payload(npes, blk)
    w.alltoall(d, s, blk)
    yield "c3a_alltoall_8x4KiB", digest(w.view(d, npes * blk))
    # C4 shape, RMAT scale 12: degrees and claimed-or-not pattern (schedule independent)
    g = configs.c4_graph(scale=12, edge_factor=16, npes=32)
    vpp, E = g.verts_per_pe, len(g.u)
    w = orc.OracleWorld(g.npes, 2 * vpp * 8 + 512)
    od, op = w.malloc(vpp * 8), w.malloc(vpp * 8)
    w.view(op, vpp * 8, np.uint64)[:] = np.uint64((1 << 64) - 1)
    w.atomic_fetch_add_batch(od, g.owner(g.u), g.local(g.u), np.ones(E, dtype=np.uint64))
    w.atomic_compare_swap_batch(op, g.owner(g.v), g.local(g.v), np.full(E, (1 << 64) - 1, dtype=np.uint64), g.u.astype(np.uint64))
    yield "c4_rmat12_degrees", digest(w.view(od, vpp * 8))
    yield "c4_rmat12_parents_sequential_schedule", digest(w.view(op, vpp * 8))
    # C5 shape, 16 PEs x 4096 elements
    npes, n = 16, 4096
    w = orc.OracleWorld(npes, 8 * n * 8)
    sf, si, d = w.malloc(n * 4), w.malloc(n * 8), w.malloc(n * 8)
    w.view(sf, n * 4, np.float32)[:] = gen.normal_f32(npes * n, 4, 0).reshape(npes, n)
    w.view(si, n * 8, np.int64)[:] = gen.uniform_i64(npes * n, -(1 << 20), 1 << 20, 4, 1).reshape(npes, n)
    w.sum_reduce_f32(d, sf, n)
    yield "c5_sum_reduce_f32_16x4096", digest(w.view(d, n * 4))
    w.sum_reduce_i64(d, si, n)
    yield "c5_sum_reduce_i64_16x4096", digest(w.view(d, n * 8))
    fc = w.malloc(npes * 256)
    w.fcollect(fc, si, 256)
    yield "c5_fcollect_16x256B", digest(w.view(fc, npes * 256))
    # C2 shape, B = 8, three rounds: ghosts and U
    h = configs.Halo(8)
    prog = h.program(with_consume=False)
    hb = sum((b + 255) // 256 * 256 for b in prog.obj_bytes) + 256
    w = orc.OracleWorld(8, hb)
    w.load_program(prog)
    for r in range(1, 4):
        U, send = w.obj("U", np.float64), w.obj("send", np.float64).reshape(8, 6, 64)
        for p in range(8):
            orc.halo_perturb(U[p], 8, h.coord(p), h.seed, r)
            for f in range(6):
                orc.halo_pack(U[p], 8, f, send[p, f])
        w.run_program(h.round_ops(prog, r, False))
    yield "c2_halo_B8_3rounds_ghost", digest(w.obj("ghost"))
    yield "c2_halo_B8_3rounds_U", digest(w.obj("U"))


def main():
    lines = ["# written by tests/golden/make_golden.py from oracle/ only; see that file's header",
             "# the paper prints no numeric example (PAPER.md L510): these pin the oracle against itself over time"]
    lines += ["%s %s" % kv for kv in cases()]
    with open(OUT, "w") as f:
        f.write("\n".join(lines) + "\n")
    print("\n".join(lines))


if __name__ == "__main__":
    main()
