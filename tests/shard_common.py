"""One seeded test case for the sharded world (NEXT-4 (iii)), written once and driven two ways: with all shards in ONE process
(worlds attached by pointer) and with one PROCESS per shard (CUDA IPC, gloo for the bootstrap).  `Case` holds what every shard
must agree on (objects, op phases, AMO streams); `ShardRunner` issues the ops a given set of local shards initiates;
`check_shard` compares what a shard holds with the rows of the GLOBAL oracle world the placement gives it."""
from __future__ import annotations

import numpy as np
import torch

from oracle import oracle as orc
from paper_2607_08006_b200 import CMP, OP, World
from workloads import gen
from workloads.spec import SIGNAL_ADD, SIGNAL_SET, Program

M64 = (1 << 64) - 1
DEV = "cuda:0"


class Case:
    def __init__(self, G: int, L: int, seed: int = 5):
        self.G, self.L, self.NP = G, L, G * L
        NP = self.NP
        rng = np.random.default_rng(seed)
        self.src_bytes, self.slot, self.nrand = 24000, 6000, 40
        self.blk = 5000                                   # alltoall block: not a multiple of 16
        self.nwords = 64
        p = Program(NP)
        p.obj("src", self.src_bytes, gen.u64(NP * self.src_bytes // 8, 91).view(np.uint8).reshape(NP, self.src_bytes))
        p.obj("dst", self.nrand * self.slot)
        p.obj("ps", NP * 10000)                           # put_signal payloads, one 10 000-byte block per sender
        p.obj("sig", 16 * NP)
        p.obj("words", 8 * self.nwords)                   # atomic add targets
        p.obj("cnt", 8 * self.nwords)                     # fetch-add(1) targets
        p.obj("par", 8 * self.nwords, np.full((NP, 8 * self.nwords), 255, dtype=np.uint8))   # compare-swap slots, init -1
        p.obj("a2a_src", NP * self.blk, gen.u64(NP * NP * self.blk // 8, 92).view(np.uint8).reshape(NP, NP * self.blk))
        p.obj("a2a_dst", NP * self.blk)
        self.blk2 = 48 * 1024 + 16                        # aligned blocks: the bulk-copy form, a ragged second chunk
        p.obj("a2b_src", NP * self.blk2, gen.u64(NP * NP * self.blk2 // 8, 93).view(np.uint8).reshape(NP, NP * self.blk2))
        p.obj("a2b_dst", NP * self.blk2)
        # collectives over all global PEs: fp32 / int64 sum_reduce (ragged share per shard), fcollect of an odd block size
        self.nred, self.fcb = 3000 + 17, 1001
        p.obj("rf_src", 4 * self.nred, gen.normal_f32(NP * self.nred, 94).view(np.uint8).reshape(NP, 4 * self.nred))
        p.obj("rf_dst", 4 * self.nred)
        p.obj("ri_src", 8 * self.nred, gen.uniform_i64(NP * self.nred, -(1 << 62), 1 << 62, 95).view(np.uint8).reshape(NP, 8 * self.nred))
        p.obj("ri_dst", 8 * self.nred)
        p.obj("fc_src", self.fcb + 7, gen.u64(NP * (self.fcb + 7 + 7) // 8 + NP, 96).view(np.uint8)[:NP * (self.fcb + 7)].reshape(NP, self.fcb + 7))
        p.obj("fc_dst", NP * self.fcb)
        self.prog = p
        # phase 1: race-free random puts / gets, any size and alignment, op k owns slot k of `dst` on the PE it writes
        ph1 = p.fork()
        for k in range(self.nrand):
            i, t = int(rng.integers(NP)), int(rng.integers(NP))
            n = int(rng.integers(0, self.slot - 40))
            s, d = int(rng.integers(0, self.src_bytes - n)), k * self.slot + int(rng.integers(0, 32))
            (ph1.put if k % 2 else ph1.get)(i, t, ("dst", d), ("src", s), n)
        # phase 2: every PE sends a payload with a signal to its right neighbour (SET) and a counted one to PE 0 (ADD)
        ph2 = p.fork()
        for i in range(NP):
            ph2.put_signal(i, (i + 1) % NP, ("ps", i * 10000), ("src", 16 * i), 9999, ("sig", 16 * i), 7 + i, SIGNAL_SET)
            ph2.put_signal(i, 0, ("ps", i * 10000 + 9999), ("src", 3), 1, ("sig", 8), 3, SIGNAL_ADD)
        # phase 3: the receivers wait (the signals are there already: the phases are separated by a barrier of the shards)
        ph3 = p.fork()
        for i in range(NP):
            ph3.signal_wait_until(i, ("sig", 16 * ((i - 1) % NP)), CMP.EQ, 7 + (i - 1) % NP)
        ph3.signal_wait_until(0, ("sig", 8), CMP.GE, 3 * NP)
        self.phases = [ph1, ph2, ph3]
        # AMO streams, one per shard (every shard issues its own stream; targets are GLOBAL PEs)
        n = 5000
        self.amo = []
        for s in range(G):
            r = np.random.default_rng(100 + s)
            self.amo.append(dict(tgt=r.integers(0, NP, n).astype(np.int32), idx=r.integers(0, self.nwords, n).astype(np.int64),
                                 val=r.integers(1, 1000, n).astype(np.uint64),
                                 claim=((np.uint64(s) << np.uint64(32)) | np.arange(n, dtype=np.uint64))))

    def heap_bytes(self):
        return sum((b + 255) // 256 * 256 for b in self.prog.obj_bytes) + 4096

    def oracle(self):
        """The GLOBAL world, every phase in order (AMO batches of the shards one after the other: adds commute)."""
        ow = orc.OracleWorld(self.NP, self.heap_bytes())
        ow.load_program(self.prog)
        for ph in self.phases:
            ow.run_program(ph)
        for a in self.amo:
            ow.atomic_add_batch(ow.objs["words"][0], a["tgt"], a["idx"], a["val"])
            ow.atomic_fetch_add_batch(ow.objs["cnt"][0], a["tgt"], a["idx"], np.ones(len(a["idx"]), dtype=np.uint64))
        ow.alltoall(ow.objs["a2a_dst"][0], ow.objs["a2a_src"][0], self.blk)
        ow.alltoall(ow.objs["a2b_dst"][0], ow.objs["a2b_src"][0], self.blk2)
        ow.sum_reduce_f32(ow.objs["rf_dst"][0], ow.objs["rf_src"][0], self.nred)
        ow.sum_reduce_i64(ow.objs["ri_dst"][0], ow.objs["ri_src"][0], self.nred)
        ow.fcollect(ow.objs["fc_dst"][0], ow.objs["fc_src"][0] + 3, self.fcb)         # unaligned source
        return ow


class ShardRunner:
    """One shard's world plus what it issues.  `off[name]` = symmetric offset (identical on every shard by construction)."""

    def __init__(self, case: Case, shard: int):
        self.case, self.shard = case, shard
        self.w = World(case.L, case.heap_bytes(), DEV)
        self.off = {}
        for name, nb in zip(case.prog.obj_names, case.prog.obj_bytes):
            o = self.w.malloc(nb)
            self.off[name] = o
            v = self.w.view(o, nb)
            if name in case.prog.init:
                v.copy_(torch.from_numpy(np.ascontiguousarray(case.prog.init[name][shard::case.G])))
            else:
                v.zero_()
        torch.cuda.synchronize()
        self.fetched = {}

    def _o(self, ops, obj_field, off_field, k):
        return self.off[self.case.prog.obj_names[int(ops[obj_field][k])]] + int(ops[off_field][k])

    def run_phase(self, ph):
        """Issue, in program order, the ops of `ph` whose initiator lives on this shard."""
        ops, w, G = ph.ops, self.w, self.case.G
        for k in range(len(ops)):
            ini, tgt, kind = int(ops["initiator"][k]), int(ops["target"][k]), int(ops["kind"][k])
            if ini % G != self.shard:
                continue
            n = int(ops["nbytes"][k])
            if kind == OP.PUT:
                w.gput(self._o(ops, "rem_obj", "rem_off", k), self._o(ops, "loc_obj", "loc_off", k), n, ini, tgt)
            elif kind == OP.GET:
                w.gget(self._o(ops, "loc_obj", "loc_off", k), self._o(ops, "rem_obj", "rem_off", k), n, ini, tgt)
            elif kind == OP.PUT_SIGNAL:
                w.gput_signal(self._o(ops, "rem_obj", "rem_off", k), self._o(ops, "loc_obj", "loc_off", k), n,
                              self._o(ops, "sig_obj", "sig_off", k), int(ops["value"][k]), int(ops["sig_op"][k]), ini, tgt)
            elif kind == OP.SIGNAL_WAIT_UNTIL:
                w.gsignal_wait_until(self._o(ops, "loc_obj", "loc_off", k), int(ops["cmp"][k]), int(ops["value"][k]), ini)
            else:
                raise AssertionError(kind)

    def run_amos(self):
        a, w = self.case.amo[self.shard], self.w
        dv = lambda x: torch.from_numpy(np.ascontiguousarray(x)).to(DEV)      # noqa: E731
        tgt, idx = dv(a["tgt"]), dv(a["idx"])
        n = len(a["idx"])
        f1 = torch.empty(n, dtype=torch.int64, device=DEV)
        f2 = torch.empty(n, dtype=torch.int64, device=DEV)
        w.gatomic_batch(OP.ATOMIC_ADD, self.off["words"], tgt, idx, val=dv(a["val"].view(np.int64)))
        w.gatomic_batch(OP.ATOMIC_FETCH_ADD, self.off["cnt"], tgt, idx.to(torch.int32), val_scalar=1, fetched_out=f1)
        w.gatomic_batch(OP.ATOMIC_COMPARE_SWAP, self.off["par"], tgt, idx, val=dv(a["claim"].view(np.int64)), cond_scalar=M64,
                        fetched_out=f2)
        self.fetched = dict(fadd=f1, cas=f2)

    def run_alltoall(self):
        self.w.galltoall(self.off["a2a_dst"], self.off["a2a_src"], self.case.blk)
        self.w.galltoall(self.off["a2b_dst"], self.off["a2b_src"], self.case.blk2)
        self.w.gsum_reduce(0, self.off["rf_dst"], self.off["rf_src"], self.case.nred)     # SHMEMG_F32
        self.w.gsum_reduce(1, self.off["ri_dst"], self.off["ri_src"], self.case.nred)     # SHMEMG_I64
        self.w.gfcollect(self.off["fc_dst"], self.off["fc_src"] + 3, self.case.fcb)

    def rows(self, name):
        return self.w.view(self.off[name], self.case.prog.obj_bytes[self.case.prog.obj_names.index(name)]).cpu().numpy()

    def results(self):
        """Everything the joint check needs from this shard, as numpy arrays."""
        out = {n: self.rows(n) for n in self.case.prog.obj_names}
        out["fetched_fadd"] = self.fetched["fadd"].cpu().numpy().view(np.uint64)
        out["fetched_cas"] = self.fetched["cas"].cpu().numpy().view(np.uint64)
        return out


def check(case: Case, results: list):
    """results[s] = ShardRunner.results() of shard s.  Bit-exact against the global oracle where the result is unique;
    invariants for the fetched values and the compare-swap winners (two shards race for the same words)."""
    ow = case.oracle()
    G, NP, nw = case.G, case.NP, case.nwords
    for s in range(G):
        for name in ("src", "dst", "ps", "sig", "words", "cnt", "a2a_src", "a2a_dst", "a2b_src", "a2b_dst", "rf_dst", "ri_dst",
                     "fc_dst"):
            off, nb = ow.objs[name]
            assert np.array_equal(results[s][name], orc.shard_rows(ow, s, G, off, nb)), (name, "shard", s)
    # global views of cnt / par assembled from the shards through the placement
    def glob(name):
        out = np.empty((NP, 8 * nw), dtype=np.uint8)
        for s in range(G):
            out[s::G] = results[s][name]
        return out.view(np.uint64)
    key = np.concatenate([a["tgt"].astype(np.int64) * nw + a["idx"] for a in case.amo])
    # fetch-add(1): over BOTH shards' ops, the fetched values of a word are a permutation of 0 .. k-1
    f = np.concatenate([results[s]["fetched_fadd"] for s in range(G)]).astype(np.int64)
    k = np.bincount(key, minlength=NP * nw)
    assert np.array_equal(glob("cnt").reshape(-1).astype(np.int64), k)
    order = np.lexsort((f, key))
    ks, fs = key[order], f[order]
    first = np.r_[0, np.flatnonzero(np.diff(ks)) + 1]
    rank = np.arange(len(ks)) - np.repeat(first, np.diff(np.r_[first, len(ks)]))
    assert np.array_equal(fs, rank), "fetched values of a word are not 0 .. k-1"
    # compare-swap(-1 -> claim): exactly one winner per touched slot, the slot holds its claim, every loser fetched the final value
    fc = np.concatenate([results[s]["fetched_cas"] for s in range(G)])
    claim = np.concatenate([a["claim"] for a in case.amo])
    par = glob("par").reshape(-1)
    won = fc == np.uint64(M64)
    assert np.array_equal(np.bincount(key[won], minlength=NP * nw), (k > 0).astype(np.int64)), "slot not claimed exactly once"
    assert np.array_equal(par[key[won]], claim[won]) and np.array_equal(fc[~won], par[key[~won]])
    assert (par[k == 0] == np.uint64(M64)).all()
