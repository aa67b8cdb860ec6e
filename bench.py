#!/usr/bin/env python
"""bench.py -- the hot-path benchmark of the B200-native GPU-aware OpenSHMEM library.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference]

One STEP is one pass of the whole hot path (every row of SURVEY.md 8(a)) over the five seeded synthetic workloads of
BASELINE.json (C1 atomic adds, C2 halo exchange x50 rounds, C3 alltoall uniform + Zipf-skewed, C4 RMAT fetch-add +
compare-swap, C5 sum_reduce / fcollect / 10 000 barriers), enqueued through the C-ABI on one stream.  Every library
call is bracketed by CUDA events on the launching stream ("segments"); application compute of the halo workload
(perturb, pack) and the re-initialisation of AMO targets run between segments and are not library time.

  metric `rma_alltoall_GBps` : algorithmic bytes of the copy-class segments (put / put_signal / alltoall / fcollect /
                               sum_reduce; read + write) / their summed device time, summed over ranks; the 50 halo rounds
                               are replayed from one CUDA graph (one event pair around 50 back-to-back launches)
  `amo_mops`                 : AMO ops of C1 + C4 / their summed device time
  `barrier`                  : us per barrier, in-kernel (128 co-resident PE agents) and stream-level
  `roofline`                 : the copy-class kernel with the largest share of the timed step, against MEASURED_PEAKS.json
  `e2e`                      : the same metric with every input copied from pinned HOST memory and every result read
                               back to the host inside the timed region (shmemg_heap_write/read_on_stream); `value`
                               pipelines upload / library call / read-back over three streams, `serial` does not
  `cpu_baseline`             : the CPU oracle (oracle/, single thread) on a bounded sample of the same workload

`--impl reference` times the oracle alone (this tier's reference arm).  N > 1 runs N independent replicas (the path
does not shard: north_star "no sharding and no inter-GPU transport"), one process per GPU, max-over-ranks timing.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

METRIC, UNIT = "rma_alltoall_GBps", "GB/s"
WORKLOAD = ("C1-C5 of BASELINE.json in one step: C3a alltoall 64 PEs x 64 KiB blocks; C3b 4096 Zipf(1.1) puts; "
            "C2 halo 8 PEs x 6 faces x 512 KiB put_signal+wait x 50 rounds; C5 sum_reduce f32/i64 + fcollect on 128 PEs "
            "+ 10 000 barriers; C1 65 536 atomic adds; C4 RMAT scale 22, 2^26 fetch-add + 2^26 compare-swap")
HALO_ROUNDS = 50
BARRIERS = 10000
M64 = (1 << 64) - 1

def ncu_traffic():
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of each copy-class segment's kernel, from the committed
    `ncu --set full` capture summarised in profiles/ (TRAFFIC_CSV; the .md beside it names the command).  Cold L2 at launch,
    up to 126 MB of the kernel's own writes still in L2 at its end, so write traffic < algorithmic writes; the halo faces are
    L2-resident by nature."""
    out = {}
    try:
        for ln in open(os.path.join(ROOT, "profiles", TRAFFIC_CSV)):
            f = [x.strip() for x in ln.split(",")]
            if len(f) >= 4 and f[0] and f[0] != "segment" and not f[0].startswith("#"):
                out[f[0]] = int(f[2]) + int(f[3])
    except OSError:
        pass
    return out


TRAFFIC_CSV = "r02_traffic.csv"


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--no-e2e", action="store_true", help="skip the end-to-end (host buffers) leg")
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg (and the verification against the oracle)")
    ap.add_argument("--no-verify", action="store_true", help="skip the comparison of every segment's results with the oracle")
    ap.add_argument("--small", action="store_true", help="reduced sizes (development only; marked in the JSON)")
    ap.add_argument("--only", default="", help="comma-separated segment groups to run: c1,c2,c3a,c3b,c4,c5,barrier,next2,next4")
    return ap.parse_args()


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "MEASURED_PEAKS.json (measured)"
        except Exception:
            pass
    return 6650.0, "B200_PROFILING.md fallback"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 100 ms while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.proc = index, None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except OSError:
            self.proc = None

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            out, _ = self.proc.communicate(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
            out, _ = self.proc.communicate()
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in out.strip().splitlines():
            f = [x.strip() for x in line.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1])); pw.append(float(f[2]))
            except ValueError:
                continue
            for n, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        return {"sm_mhz": statistics.median(sm), "sm_max_mhz": max(mx), "power_w_max": max(pw), "samples": len(sm),
                "reasons": sorted(reasons)}


# ======================================================================================================================
# inputs: generated once on the host by the seeded generators of workloads/ (no method arithmetic there)
# ======================================================================================================================
class Inputs:
    def __init__(self, small: bool, groups):
        from workloads import configs
        self.small = small
        t0 = time.time()
        self.groups = groups
        if "c1" in groups:
            self.c1 = configs.c1_atomic_add()
            self.c1_steady = configs.c1_atomic_add(n_ops=(1 << 18) if small else (1 << 24))   # same distribution
        if "c2" in groups:
            self.halo = configs.Halo(64 if small else 256)
            self.halo_U = self.halo.initial_U()
        if "c3a" in groups:
            self.c3a_npes, self.c3a_blk = (16, 65536) if small else (64, 65536)
            self.c3a = configs.c3a_payload(self.c3a_npes, self.c3a_blk)
        if "c3b" in groups:
            self.c3b = configs.c3b_skewed(npes=16 if small else 64)
        if "c4" in groups:
            self.c4 = configs.c4_graph(scale=18 if small else 22)
        if "next4" in groups:
            # NEXT-4 (i): slab transpose of a 1024 x 1024 x 256 complex64 array (2 GiB) over 64 PEs
            self.fft = configs.fft_transpose(16, 128, 128, 64) if small else configs.fft_transpose()
            # NEXT-4 (iii): the C3a alltoall on a world sharded over TWO worlds (both on this one GPU, attached by pointer)
            self.sh_npes, self.sh_blk = (16, 65536) if small else (64, 65536)
            self.sh_payload = getattr(self, "c3a", None)
            if self.sh_payload is None or self.sh_payload.shape[0] != self.sh_npes:
                self.sh_payload = configs.c3a_payload(self.sh_npes, self.sh_blk)
        if "c5" in groups or "barrier" in groups:
            self.c5_npes, self.c5_bytes = (32, 1 << 20) if small else (128, 4 << 20)
            self.c5_fc_bytes = 32768
        if "c5" in groups:
            self.c5_f32 = configs.c5_f32(self.c5_npes, self.c5_bytes // 4)
            self.c5_i64 = configs.c5_i64(self.c5_npes, self.c5_bytes // 8)
            self.c5_fc = configs.c5_fcollect_src(self.c5_npes, self.c5_fc_bytes)
        self.gen_seconds = time.time() - t0


# algorithmic bytes / ops of each segment: copies count read + write
def segment_table(inp: Inputs):
    seg = {}
    g = inp.groups
    if "c3a" in g:
        n, b = inp.c3a_npes, inp.c3a_blk
        seg["alltoall"] = dict(cls="copy", kernel="k_alltoall_tma", bytes=2 * n * n * b, launches=1)
    if "c3b" in g:
        seg["put_batch_skewed"] = dict(cls="copy", kernel="k_batch_exec", bytes=2 * int(inp.c3b.sizes.sum()), launches=1)
    if "c2" in g:
        # the 50 pre-planned rounds replayed from ONE CUDA graph (the launch-bound inner loop of the application), one event
        # pair around the replay: 50 back-to-back launches of k_batch_exec, nothing else in the timed region
        seg["halo_put_signal_wait"] = dict(cls="copy", kernel="k_batch_exec", l2_resident=True,
                                           bytes=HALO_ROUNDS * 2 * 48 * inp.halo.face_bytes, launches=HALO_ROUNDS)
        # the same 50 launches enqueued one by one from the host between the application's kernels, an event pair around
        # EACH launch (round 1's measurement; an event pair around any kernel costs about 6 us whatever the kernel does)
        seg["halo_put_signal_wait_event_pairs"] = dict(cls="xcopy", kernel="k_batch_exec",
                                                       bytes=HALO_ROUNDS * 2 * 48 * inp.halo.face_bytes, launches=HALO_ROUNDS)
    # the ONE-CALL form of the two batch workloads (shmemg_enqueue_batch: device-resident descriptors planned on the device
    # inside the timed segment, 2 launches); reported beside the pre-planned form, not part of `value`
    if "c3b" in g:
        seg["put_batch_skewed_onecall"] = dict(cls="xcopy", kernel="k_plan_batch + k_batch_exec", bytes=2 * int(inp.c3b.sizes.sum()), launches=1)
    if "c2" in g:
        seg["halo_put_signal_wait_onecall"] = dict(cls="xcopy", kernel="k_plan_batch + k_batch_exec",
                                                   bytes=HALO_ROUNDS * 2 * 48 * inp.halo.face_bytes, launches=HALO_ROUNDS)
    if "c2" in g:
        # the 50 one-call rounds replayed from ONE CUDA graph (device planner + executor per round, back to back)
        seg["halo_put_signal_wait_onecall_graph"] = dict(cls="xcopy", kernel="k_plan_batch + k_batch_exec",
                                                         bytes=HALO_ROUNDS * 2 * 48 * inp.halo.face_bytes, launches=HALO_ROUNDS)
    if "c5" in g:
        n, nb = inp.c5_npes, inp.c5_bytes
        seg["sum_reduce_f32"] = dict(cls="copy", kernel="k_sum_reduce_tma<f32>", bytes=2 * n * nb, launches=1)
        seg["sum_reduce_i64"] = dict(cls="copy", kernel="k_sum_reduce_tma<i64>", bytes=2 * n * nb, launches=1)
        seg["fcollect"] = dict(cls="copy", kernel="k_fcollect_tma",
                               bytes=n * inp.c5_fc_bytes + n * n * inp.c5_fc_bytes, launches=1)
    if "c1" in g:
        # operand / result streams per op (what HBM must move): C1 tgt_pe 4 + idx 8 + val 8
        seg["atomic_add"] = dict(cls="amo", kernel="k_amo<add> (quiet + barrier folded into the launch)", ops=len(inp.c1.val),
                                 launches=1, bytes_per_op=20)
        # the same distribution, 2^24 ops: the kernel's steady-state rate (reported, not part of `amo_mops`)
        seg["atomic_add_steady_2p24"] = dict(cls="xamo", kernel="k_amo<add>", ops=len(inp.c1_steady.val), launches=1, bytes_per_op=20)
    if "c4" in g:
        E = len(inp.c4.u)
        # fetch-add: tgt_pe 4 + idx 4 read, 8 fetched written; plain compare-swap: tgt_pe 4 + idx 4 + val 8 read, 8 fetched written
        seg["atomic_fetch_add"] = dict(cls="amo", kernel="k_hot_sample + k_amo_hot_main<fetch_add>", ops=E, launches=2, bytes_per_op=16)
        # test-before-swap, streaming form: tgt_pe 4 + idx 4 read, 8 fetched written; val (8) is read only by the ops that issue the atomic
        seg["atomic_compare_swap"] = dict(cls="amo", kernel="k_cas_test (test-before-swap, L1-served test loads, lazy val)", ops=E, launches=1, bytes_per_op=16)
        # every op an L2 atomic (no test load): the variant the atom.cas ceiling bounds; reported, not part of `amo_mops`
        seg["atomic_compare_swap_plain"] = dict(cls="xamo", kernel="k_amo<compare_swap>", ops=E, launches=1, bytes_per_op=24)
    if "next2" in g:
        # NEXT-2 surface; reported per segment, NOT part of `value` / `amo_mops` (cls x*)
        if "c5" in g:
            n, nb = inp.c5_npes, inp.c5_bytes
            seg["next2_broadcast"] = dict(cls="xcopy", kernel="k_broadcast_tma", bytes=(n + 1) * nb, launches=1)
            seg["next2_reduce_max_i64"] = dict(cls="xcopy", kernel="k_sum_reduce_tma<i64,max>", bytes=2 * n * nb, launches=1)
            seg["next2_reduce_min_f32"] = dict(cls="xcopy", kernel="k_sum_reduce_tma<f32,min>", bytes=2 * n * nb, launches=1)
            # NEXT-1: the same fp32 sum_reduce as a DEVICE collective (one thread block per PE calls shmemg_dev_sum_reduce_block)
            seg["next1_dev_sum_reduce_f32"] = dict(cls="xcopy", kernel="k_device_collective (shmemg_dev_sum_reduce_block)", bytes=2 * n * nb, launches=1)
        if "c4" in g:
            seg["next2_amo_xor"] = dict(cls="xamo", kernel="k_amo2<xor>", ops=len(inp.c4.u), launches=1)
            seg["next2_amo_fetch_xor"] = dict(cls="xamo", kernel="k_amo2<fetch_xor>", ops=len(inp.c4.u), launches=1)
        if "c2" in g:
            # NEXT-1: the whole halo APPLICATION (compute + exchange) per round, three ways; us per round is what counts
            seg["next1_halo_app_host_batches"] = dict(cls="xtime", kernel="k_halo_perturb + k_halo_pack + k_batch_exec", ops=HALO_ROUNDS, launches=3 * HALO_ROUNDS)
            seg["next1_halo_app_persistent"] = dict(cls="xtime", kernel="k_halo_persistent (device-initiated)", ops=HALO_ROUNDS, launches=1)
            seg["next1_halo_app_compute_only"] = dict(cls="xtime", kernel="k_halo_perturb", ops=HALO_ROUNDS, launches=HALO_ROUNDS)
            # the application loop from a CUDA graph, with and without the library's launches: the difference is what a
            # round of put_signal + wait adds to the application's critical path
            seg["next1_halo_app_graph"] = dict(cls="xtime", kernel="graph: k_halo_perturb + k_halo_pack + k_batch_exec", ops=HALO_ROUNDS, launches=3 * HALO_ROUNDS)
            seg["next1_halo_app_graph_without_exchange"] = dict(cls="xtime", kernel="graph: k_halo_perturb + k_halo_pack", ops=HALO_ROUNDS, launches=2 * HALO_ROUNDS)
            seg["next2_ibput_faces"] = dict(cls="xcopy", kernel="k_ib_tma/k_ib_elem", bytes=3 * 2 * inp.halo.face_bytes, launches=3)
    if "next4" in g:
        seg["next4_fft_transpose_alltoalls"] = dict(cls="xcopy", kernel="k_alltoalls_tma", bytes=2 * inp.fft.A.size, launches=1)
        seg["next4_sharded_alltoall_2_shards_on_one_gpu"] = dict(cls="xcopy", kernel="k_shard_alltoall (one launch per shard)",
                                                                 bytes=2 * inp.sh_npes ** 2 * inp.sh_blk, launches=2)
    if "barrier" in g:
        seg["barrier_in_kernel"] = dict(cls="sync", kernel="k_barrier_repeat", ops=BARRIERS, launches=1)
        seg["barrier_on_stream"] = dict(cls="sync", kernel="k_barrier_epoch", ops=BARRIERS, launches=BARRIERS)
        seg["barrier_on_stream_graph"] = dict(cls="sync", kernel="k_barrier_epoch", ops=BARRIERS, launches=BARRIERS)
    return seg


# ======================================================================================================================
# CUDA arm: everything goes through the C-ABI (binding = argument marshalling only)
# ======================================================================================================================
class _Null:
    def __enter__(self):
        return self

    def __exit__(self, *exc):
        return False


class Recorder:
    """CUDA-event pairs around library calls, on the launching (current) stream."""

    def __init__(self, torch):
        self.torch, self.pairs, self.on = torch, [], False

    class _Seg:
        def __init__(self, rec, name):
            self.rec, self.name = rec, name

        def __enter__(self):
            if self.rec.on:
                self.a = self.rec.torch.cuda.Event(enable_timing=True)
                self.b = self.rec.torch.cuda.Event(enable_timing=True)
                self.a.record()

        def __exit__(self, *exc):
            if self.rec.on:
                self.b.record()
                self.rec.pairs.append((self.name, self.a, self.b))

    def seg(self, name):
        return Recorder._Seg(self, name)

    def totals_ms(self):
        out = {}
        for name, a, b in self.pairs:
            out[name] = out.get(name, 0.0) + a.elapsed_time(b)
        return out


class CudaBench:
    def __init__(self, inp: Inputs, device):
        import torch
        from paper_2607_08006_b200 import World
        from paper_2607_08006_b200.binding import AMO_HOT_AGGREGATE, AMO_TEST_BEFORE_SWAP, AMO_THEN_BARRIER
        self.c1_flags = AMO_THEN_BARRIER               # C1 ends with quiet + barrier: folded into the AMO launch
        from paper_2607_08006_b200.loader import Loaded
        self.torch, self.inp, self.dev = torch, inp, device
        self.rec = Recorder(torch)
        self.app_launches = 0
        self.plan_us = {}                              # host planning cost of the pre-planned batches (outside every timed region)
        self.barrier_graph = None
        self.halo_graphs = None                        # CUDA graphs of the 50 halo rounds (captured in the first step)
        self.worlds = []
        self.flags = 0                                 # warp aggregation buys nothing on these streams (profiles/)
        self.fadd_flags = AMO_HOT_AGGREGATE            # RMAT stream: the hot words are combined per CTA chunk (profiles/r01d)
        self.cas_flags = AMO_TEST_BEFORE_SWAP          # scalar cond: failed swaps are resolved by a coherent load
        g = inp.groups
        dv = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(device)      # noqa: E731
        if "c3a" in g:
            n, b = inp.c3a_npes, inp.c3a_blk
            w = World(n, 2 * n * b + 4096, device)
            self.w3a, self.a_src, self.a_dst = w, w.malloc(n * b), w.malloc(n * b)
            w.view(self.a_src, n * b).copy_(torch.from_numpy(inp.c3a))
            w.view(self.a_dst, n * b).zero_()
            self.worlds.append(w)
        if "c3b" in g:
            prog = inp.c3b.prog
            hb = sum((x + 255) // 256 * 256 for x in prog.obj_bytes) + 4096
            w = World(prog.npes, hb, device)
            self.w3b, self.ld3b = w, Loaded(w, prog)
            ops = self.ld3b.translate(prog)
            t0 = time.perf_counter()
            self.b3b = w.batch(ops)                                   # shmemg_batch_plan_bytes + shmemg_batch_create (ends in a stream sync)
            self.plan_us["put_batch_skewed"] = {"nops": len(ops), "host_plan_us": (time.perf_counter() - t0) * 1e6}
            self.ops3b_host = torch.from_numpy(ops.view(np.uint8).reshape(-1).copy()).pin_memory()
            self.ops3b_dev = self.ops3b_host.to(device)
            self.work3b = torch.empty(w.batch_work_bytes(len(ops), int(inp.c3b.sizes.sum())), dtype=torch.uint8, device=device)
            self.worlds.append(w)
        if "c2" in g:
            h = inp.halo
            prog = h.program(with_consume=False, with_U=False)
            hb = h.B ** 3 * 8 + sum((x + 255) // 256 * 256 for x in prog.obj_bytes) + 8192
            w = World(8, hb, device)
            self.w2 = w
            self.U_off = w.malloc(h.B ** 3 * 8)
            w.view(self.U_off, h.B ** 3 * 8).copy_(torch.from_numpy(inp.halo_U.view(np.uint8)))
            self.ld2 = Loaded(w, prog)
            halo_ops = [self.ld2.translate(h.round_ops(prog, r, False)) for r in range(1, HALO_ROUNDS + 1)]
            self.halo_batches, ts = [], []
            for ops in halo_ops:
                t0 = time.perf_counter()
                self.halo_batches.append(w.batch(ops))
                ts.append((time.perf_counter() - t0) * 1e6)
            self.plan_us["halo_put_signal_wait"] = {"nops": len(halo_ops[0]), "host_plan_us": statistics.median(ts),
                                                    "plans": HALO_ROUNDS}
            self.halo_ops_host = [torch.from_numpy(o.view(np.uint8).reshape(-1).copy()).pin_memory() for o in halo_ops]
            self.halo_ops_dev = [t.to(device) for t in self.halo_ops_host]
            self.worlds.append(w)
        if "next4" in g:
            t = inp.fft
            w = World(t.npes, 2 * t.slab_bytes + 4096, device)
            self.wf, self.f_src, self.f_dst = w, w.malloc(t.slab_bytes), w.malloc(t.slab_bytes)
            w.view(self.f_src, t.slab_bytes).copy_(torch.from_numpy(t.A))
            w.view(self.f_dst, t.slab_bytes).zero_()
            self.worlds.append(w)
            n, b = inp.sh_npes, inp.sh_blk
            self.wsh = [World(n // 2, 2 * n * b + 4096, device) for _ in range(2)]
            for sh, ws in enumerate(self.wsh):
                ws.shard_init(2, sh)
            self.wsh[0].shard_attach_world(1, self.wsh[1])
            self.wsh[1].shard_attach_world(0, self.wsh[0])
            offs = [(ws.malloc(n * b), ws.malloc(n * b)) for ws in self.wsh]
            assert offs[0] == offs[1]                                  # the same allocations on every shard: one offset names one object
            self.sh_src, self.sh_dst = offs[0]
            for sh, ws in enumerate(self.wsh):
                ws.view(self.sh_src, n * b).copy_(torch.from_numpy(np.ascontiguousarray(inp.sh_payload[sh::2])))
                ws.view(self.sh_dst, n * b).zero_()
                self.worlds.append(ws)
        if "c5" in g or "barrier" in g:
            n, nb = inp.c5_npes, inp.c5_bytes
            w = World(n, 3 * nb + inp.c5_fc_bytes + 65536, device)
            self.w5 = w
            self.worlds.append(w)
            self.stamp = w.calloc(3, 8)
        if "c5" in g:
            w = self.w5
            self.s_f32, self.s_i64, self.d5, self.s_fc = w.malloc(nb), w.malloc(nb), w.malloc(nb), w.malloc(inp.c5_fc_bytes)
            w.view(self.s_f32, nb, torch.float32).copy_(torch.from_numpy(inp.c5_f32))
            w.view(self.s_i64, nb, torch.int64).copy_(torch.from_numpy(inp.c5_i64))
            w.view(self.s_fc, inp.c5_fc_bytes).copy_(torch.from_numpy(inp.c5_fc))
        if "c1" in g:
            c = inp.c1
            w = World(c.npes, c.nelem * 8 + 4096, device)
            self.w1, self.A = w, w.calloc(c.nelem, 8)
            self.c1_t, self.c1_i, self.c1_v = dv(c.tgt_pe), dv(c.idx.astype(np.int64)), dv(c.val)
            cs = inp.c1_steady
            self.c1s = (dv(cs.tgt_pe), dv(cs.idx.astype(np.int64)), dv(cs.val))
            self.worlds.append(w)
        if "c4" in g:
            q = inp.c4
            vpp, E = q.verts_per_pe, len(q.u)
            w = World(q.npes, 2 * vpp * 8 + 4096, device)
            self.w4, self.deg, self.par = w, w.calloc(vpp, 8), w.malloc(vpp * 8)
            self.c4_ou, self.c4_lu = dv(q.owner(q.u)), dv(q.local(q.u).astype(np.uint32).view(np.int32))
            self.c4_ov, self.c4_lv = dv(q.owner(q.v)), dv(q.local(q.v).astype(np.uint32).view(np.int32))
            self.c4_val = dv(q.u.astype(np.int64))
            self.f_deg = torch.empty(E, dtype=torch.int64, device=device)
            self.f_par = torch.empty(E, dtype=torch.int64, device=device)
            w.set_scratch_for(E)                       # caller-owned scratch of the hot-set kernels (the library allocates nothing)
            self.worlds.append(w)
        torch.cuda.synchronize(device)

    def launches(self):
        return sum(w.launches for w in self.worlds) + self.app_launches

    # ---- one pass of the whole hot path; device-resident inputs ------------------------------------------------------
    def step(self):
        """Order: the millisecond-long AMO kernels first, so the host runs ahead of the device and every later segment
        measures device time with its launch already queued (the events bracket the kernel, not host launch latency)."""
        torch, inp, rec, g = self.torch, self.inp, self.rec, self.inp.groups
        if "c4" in g:
            vpp = inp.c4.verts_per_pe
            self.w4.view(self.deg, vpp * 8).zero_()
            self.w4.view(self.par, vpp * 8).fill_(255)
            with rec.seg("atomic_fetch_add"):
                self.w4.atomic_fetch_add_batch(self.deg, self.c4_ou, self.c4_lu, self.f_deg, val=None, val_scalar=1,
                                               flags=self.fadd_flags)
            with rec.seg("atomic_compare_swap"):
                self.w4.atomic_compare_swap_batch(self.par, self.c4_ov, self.c4_lv, self.f_par, cond=None, cond_scalar=M64,
                                                  val=self.c4_val, flags=self.cas_flags)
            self.w4.view(self.par, vpp * 8).fill_(255)
            with rec.seg("atomic_compare_swap_plain"):
                self.w4.atomic_compare_swap_batch(self.par, self.c4_ov, self.c4_lv, self.f_par, cond=None, cond_scalar=M64,
                                                  val=self.c4_val, flags=0)
        if "c1" in g:
            self.w1.view(self.A, inp.c1.nelem * 8).zero_()
            with rec.seg("atomic_add"):
                self.w1.atomic_add_batch(self.A, self.c1_t, self.c1_i, val=self.c1_v, flags=self.flags | self.c1_flags)
            with rec.seg("atomic_add_steady_2p24"):
                self.w1.atomic_add_batch(self.A, *self.c1s[:2], val=self.c1s[2], flags=self.flags)
        if "c3a" in g:
            with rec.seg("alltoall"):
                self.w3a.alltoall(self.a_dst, self.a_src, inp.c3a_blk)
        if "c5" in g:
            n = inp.c5_bytes
            with rec.seg("sum_reduce_f32"):
                self.w5.sum_reduce(0, self.d5, self.s_f32, n // 4)
        if "c3b" in g:
            with rec.seg("put_batch_skewed"):
                self.w3b.enqueue_batch(self.b3b)
        if "c5" in g:
            with rec.seg("sum_reduce_i64"):
                self.w5.sum_reduce(1, self.d5, self.s_i64, n // 8)
            with rec.seg("fcollect"):
                self.w5.fcollect(self.d5, self.s_fc, inp.c5_fc_bytes)
        if "c2" in g:
            h, w = inp.halo, self.w2
            self.ld2.obj("sig").zero_()                                  # rounds restart at 1 every step
            send_off = self.ld2.off["send"][0]
            with rec.seg("next1_halo_app_host_batches") if "next2" in g else _Null():
                for r in range(1, HALO_ROUNDS + 1):
                    w.app_halo_perturb(self.U_off, h.B, h.seed, r)       # application compute, not library time
                    w.app_halo_pack(send_off, self.U_off, h.B)
                    self.app_launches += 2
                    with rec.seg("halo_put_signal_wait_event_pairs"):
                        w.enqueue_batch(self.halo_batches[r - 1])
            if self.halo_graphs is None:
                self.halo_graphs = self._capture_halo_graphs()
            lib_g, app_g, app_only_g, onecall_g = self.halo_graphs
            self.ld2.obj("sig").zero_()
            w.app_halo_pack(send_off, self.U_off, h.B)                   # faces as the application leaves them (outside the timed region)
            self.app_launches += 1
            with rec.seg("halo_put_signal_wait"):
                lib_g.replay()
            w.launches += HALO_ROUNDS
            self.ld2.obj("sig").zero_()
            with rec.seg("halo_put_signal_wait_onecall_graph"):
                onecall_g.replay()
            w.launches += 2 * HALO_ROUNDS
            if "next2" in g:
                with rec.seg("next1_halo_app_graph"):
                    app_g.replay()
                w.launches += HALO_ROUNDS
                with rec.seg("next1_halo_app_graph_without_exchange"):
                    app_only_g.replay()
                self.app_launches += 4 * HALO_ROUNDS
        if "c3b" in g:
            with rec.seg("put_batch_skewed_onecall"):
                self.w3b.enqueue_batch_dev(self.ops3b_dev, self.plan_us["put_batch_skewed"]["nops"], self.work3b)
        if "c2" in g:
            h, w = inp.halo, self.w2
            self.ld2.obj("sig").zero_()
            send_off = self.ld2.off["send"][0]
            for r in range(1, HALO_ROUNDS + 1):
                w.app_halo_pack(send_off, self.U_off, h.B)               # faces freshly written (L2), as in the rounds above
                self.app_launches += 1
                with rec.seg("halo_put_signal_wait_onecall"):
                    w.enqueue_batch_dev(self.halo_ops_dev[r - 1], 96)    # plan arena of the world
        if "next2" in g:
            from paper_2607_08006_b200.binding import AMO, F32, I64, RED
            if "c5" in g:
                n = inp.c5_bytes
                with rec.seg("next2_broadcast"):
                    self.w5.broadcast(self.d5, self.s_i64, n, 3)
                with rec.seg("next2_reduce_max_i64"):
                    self.w5.reduce(RED.MAX, I64, self.d5, self.s_i64, n // 8)
                with rec.seg("next2_reduce_min_f32"):
                    self.w5.reduce(RED.MIN, F32, self.d5, self.s_f32, n // 4)
                with rec.seg("next1_dev_sum_reduce_f32"):
                    self.w5.device_collective(0, self.d5, self.s_f32, n // 4, dtype=F32)
            if "c4" in g:
                with rec.seg("next2_amo_xor"):
                    self.w4.atomic_op_batch(AMO.XOR, 8, self.deg, self.c4_ou, self.c4_lu, val=self.c4_val)
                with rec.seg("next2_amo_fetch_xor"):
                    self.w4.atomic_op_batch(AMO.XOR, 8, self.deg, self.c4_ou, self.c4_lu, val=self.c4_val, fetched_out=self.f_deg)
            if "c2" in g:
                h, B = inp.halo, inp.halo.B
                self.ld2.obj("sig").zero_()
                with rec.seg("next1_halo_app_persistent"):     # the same 50 rounds in ONE device-initiated kernel
                    self.w2.app_halo_persistent(self.U_off, self.ld2.off["ghost"][0], self.ld2.off["sig"][0], B, h.seed, 1, HALO_ROUNDS)
                    self.app_launches += 1
                with rec.seg("next1_halo_app_compute_only"):
                    for r in range(1, HALO_ROUNDS + 1):
                        self.w2.app_halo_perturb(self.U_off, B, h.seed, r)
                    self.app_launches += HALO_ROUNDS
                send_off, fb = self.ld2.off["send"][0], inp.halo.face_bytes
                with rec.seg("next2_ibput_faces"):             # the three face orientations straight out of the cube
                    self.w2.ibput(send_off, self.U_off, 0, 0, fb, 1, 0, 1)
                    self.w2.ibput(send_off + 2 * fb, self.U_off, B * 8, B * B * 8, B * 8, B, 0, 1)
                    self.w2.ibput(send_off + 4 * fb, self.U_off, 8, B * 8, 8, B * B, 0, 1)
        if "next4" in g:
            block, nblocks, sbs, sps, dbs, dps = inp.fft.params()
            with rec.seg("next4_fft_transpose_alltoalls"):
                self.wf.alltoalls(self.f_dst, self.f_src, dps, sps, dbs, sbs, block, nblocks)
            with rec.seg("next4_sharded_alltoall_2_shards_on_one_gpu"):
                for ws in self.wsh:
                    ws.galltoall(self.sh_dst, self.sh_src, inp.sh_blk)
        if "barrier" in g:
            with rec.seg("barrier_in_kernel"):
                self.w5.barrier_all_repeat(BARRIERS)
            with rec.seg("barrier_on_stream"):
                for _ in range(BARRIERS):
                    self.w5.barrier_all()
            if self.barrier_graph is None:                               # the same 10 000 launches captured once (reading 24)
                self.barrier_graph = torch.cuda.CUDAGraph()
                with torch.cuda.graph(self.barrier_graph, capture_error_mode="thread_local"):   # other threads (an NCCL watchdog under torchrun) may call CUDA
                    for _ in range(BARRIERS):
                        self.w5.barrier_all()
            with rec.seg("barrier_on_stream_graph"):
                self.barrier_graph.replay()
                self.w5.launches += BARRIERS

    def _capture_halo_graphs(self):
        """Three CUDA graphs over the 50 halo rounds: the library's launches alone (back to back), the application loop
        (perturb, pack, batch) and the application loop without the exchange.  The pre-planned batches are re-enqueueable
        (monotonic counters), so a captured launch replays any number of times."""
        torch, h, w = self.torch, self.inp.halo, self.w2
        send_off, l0, a0 = self.ld2.off["send"][0], w.launches, self.app_launches
        graphs = []
        for app, lib in ((False, True), (True, True), (True, False), (False, "one-call")):
            gr = torch.cuda.CUDAGraph()
            with torch.cuda.graph(gr, capture_error_mode="thread_local"):
                if app:
                    self.ld2.obj("sig").zero_()
                for r in range(1, HALO_ROUNDS + 1):
                    if app:
                        w.app_halo_perturb(self.U_off, h.B, h.seed, r)
                        w.app_halo_pack(send_off, self.U_off, h.B)
                    if lib == "one-call":
                        w.enqueue_batch_dev(self.halo_ops_dev[r - 1], 96)
                    elif lib:
                        w.enqueue_batch(self.halo_batches[r - 1])
            graphs.append(gr)
        w.launches, self.app_launches = l0, a0                           # capturing launches nothing
        return graphs

    # ---- end-to-end: the same ops with HOST buffers, H2D / D2H inside the timed region --------------------------------
    def setup_e2e(self):
        torch, inp, g = self.torch, self.inp, self.inp.groups
        pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()      # noqa: E731
        pz = lambda *shape, dt=torch.uint8: torch.empty(*shape, dtype=dt).pin_memory()  # noqa: E731
        self.h2d = self.d2h = 0
        if "c3a" in g:
            self.h_a_src, self.h_a_dst = pin(inp.c3a), pz(*inp.c3a.shape)
        if "c3b" in g:
            self.h_b_src = pin(inp.c3b.prog.init["src"])
            self.h_b_dst = pz(inp.c3b.prog.npes, inp.c3b.dst_bytes)
        if "c2" in g:
            fb = inp.halo.face_bytes
            send = self.ld2.obj("send").cpu().contiguous()                      # faces of the last round: representative payload
            self.h_send, self.h_ghost = send.pin_memory(), pz(8, 6 * fb)
        if "c5" in g:
            self.h_f32, self.h_i64, self.h_fc = pin(inp.c5_f32.view(np.uint8)), pin(inp.c5_i64.view(np.uint8)), pin(inp.c5_fc)
            self.h_res = pz(3, inp.c5_bytes)
        if "c1" in g:
            c = inp.c1
            self.h_c1 = [pin(c.tgt_pe), pin(c.idx.astype(np.int64)), pin(c.val)]
            self.h_A = pz(c.npes, c.nelem * 8)
        if "c4" in g:
            self.h_c4 = [pin(t.cpu().numpy()) for t in (self.c4_ou, self.c4_lu, self.c4_ov, self.c4_lv, self.c4_val)]
            E = len(inp.c4.u)
            self.h_fdeg, self.h_fpar = pz(E, dt=torch.int64), pz(E, dt=torch.int64)
            self.h_deg, self.h_par = pz(inp.c4.npes, inp.c4.verts_per_pe * 8), pz(inp.c4.npes, inp.c4.verts_per_pe * 8)

    def _up(self, w, off, host2d):
        for p in range(host2d.shape[0]):
            w.heap_write(p, off, host2d[p])
        self.h2d += host2d.numel() * host2d.element_size()

    def _down(self, w, host2d, off):
        for p in range(host2d.shape[0]):
            w.heap_read(p, host2d[p], off)
        self.d2h += host2d.numel() * host2d.element_size()

    def _e2e_segments(self):
        """The end-to-end leg as (segment, class, upload, library call, read-back) tuples: `upload` copies the segment's inputs
        from pinned host memory, `read-back` its results to pinned host memory; all three enqueue on torch's CURRENT stream."""
        inp, g, out = self.inp, self.inp.groups, []

        def cp_in(dev_t, host_t):
            dev_t.copy_(host_t, non_blocking=True)
            self.h2d += host_t.numel() * host_t.element_size()

        def cp_out(host_t, dev_t):
            host_t.copy_(dev_t, non_blocking=True)
            self.d2h += host_t.numel() * host_t.element_size()
        if "c3a" in g:
            out.append(("alltoall", "copy", lambda: self._up(self.w3a, self.a_src, self.h_a_src),
                        lambda: self.w3a.alltoall(self.a_dst, self.a_src, inp.c3a_blk),
                        lambda: self._down(self.w3a, self.h_a_dst, self.a_dst)))
        if "c3b" in g:                                                   # descriptors are host inputs too: one-call form
            out.append(("put_batch_skewed", "copy",
                        lambda: (self._up(self.w3b, self.ld3b.off["src"][0], self.h_b_src), cp_in(self.ops3b_dev, self.ops3b_host)),
                        lambda: self.w3b.enqueue_batch_dev(self.ops3b_dev, self.plan_us["put_batch_skewed"]["nops"], self.work3b),
                        lambda: self._down(self.w3b, self.h_b_dst, self.ld3b.off["dst"][0])))
        if "c5" in g:
            n = inp.c5_bytes                                             # every PE holds the same result: PE 0's is read back
            out.append(("sum_reduce_f32", "copy", lambda: self._up(self.w5, self.s_f32, self.h_f32),
                        lambda: self.w5.sum_reduce(0, self.d5, self.s_f32, n // 4), lambda: self._down(self.w5, self.h_res[0:1], self.d5)))
            out.append(("sum_reduce_i64", "copy", lambda: self._up(self.w5, self.s_i64, self.h_i64),
                        lambda: self.w5.sum_reduce(1, self.d5, self.s_i64, n // 8), lambda: self._down(self.w5, self.h_res[1:2], self.d5)))
            out.append(("fcollect", "copy", lambda: self._up(self.w5, self.s_fc, self.h_fc),
                        lambda: self.w5.fcollect(self.d5, self.s_fc, inp.c5_fc_bytes), lambda: self._down(self.w5, self.h_res[2:3], self.d5)))
        if "c2" in g:
            w, fb = self.w2, inp.halo.face_bytes
            send_off, ghost_off = self.ld2.off["send"][0], self.ld2.off["ghost"][0]
            for r in range(1, HALO_ROUNDS + 1):
                out.append(("halo_put_signal_wait", "copy",
                            lambda r=r: (self._up(w, send_off, self.h_send), cp_in(self.halo_ops_dev[r - 1], self.halo_ops_host[r - 1])),
                            lambda r=r: ((self.ld2.obj("sig").zero_() if r == 1 else None), w.enqueue_batch_dev(self.halo_ops_dev[r - 1], 96)),
                            lambda r=r: self._down(w, self.h_ghost, ghost_off + (r & 1) * 6 * fb)))
        if "c1" in g:
            out.append(("atomic_add", "amo",
                        lambda: [cp_in(d, h) for d, h in zip((self.c1_t, self.c1_i, self.c1_v), self.h_c1)],
                        lambda: (self.w1.view(self.A, inp.c1.nelem * 8).zero_(),
                                 self.w1.atomic_add_batch(self.A, self.c1_t, self.c1_i, val=self.c1_v, flags=self.flags | self.c1_flags)),
                        lambda: self._down(self.w1, self.h_A, self.A)))
        if "c4" in g:
            vpp = inp.c4.verts_per_pe
            out.append(("atomic_fetch_add", "amo",
                        lambda: [cp_in(d, h) for d, h in zip((self.c4_ou, self.c4_lu), self.h_c4[:2])],
                        lambda: (self.w4.view(self.deg, vpp * 8).zero_(),
                                 self.w4.atomic_fetch_add_batch(self.deg, self.c4_ou, self.c4_lu, self.f_deg, val=None, val_scalar=1,
                                                                flags=self.fadd_flags)),
                        lambda: (cp_out(self.h_fdeg, self.f_deg), self._down(self.w4, self.h_deg, self.deg))))
            out.append(("atomic_compare_swap", "amo",
                        lambda: [cp_in(d, h) for d, h in zip((self.c4_ov, self.c4_lv, self.c4_val), self.h_c4[2:])],
                        lambda: (self.w4.view(self.par, vpp * 8).fill_(255),
                                 self.w4.atomic_compare_swap_batch(self.par, self.c4_ov, self.c4_lv, self.f_par, cond=None, cond_scalar=M64,
                                                                   val=self.c4_val, flags=self.cas_flags)),
                        lambda: (cp_out(self.h_fpar, self.f_par), self._down(self.w4, self.h_par, self.par))))
        return out

    def e2e_step(self):
        """Serial form: every segment's upload, library call and read-back on ONE stream inside its own event pair."""
        for name, _cls, up, call, down in self._e2e_segments():
            with self.rec.seg(name):
                up(); call(); down()

    def e2e_check(self):
        """After a pipelined step: what was read back to the host equals what the device holds (the read-backs were ordered
        behind their library calls), for every result buffer of the copy-class segments and the AMO arrays."""
        torch, g, ok = self.torch, self.inp.groups, True
        torch.cuda.synchronize()
        eq = lambda host2d, w, off: bool(torch.equal(host2d, w.view(off, host2d.shape[1])[:host2d.shape[0]].cpu()))   # noqa: E731
        if "c3a" in g:
            ok &= eq(self.h_a_dst, self.w3a, self.a_dst)
        if "c3b" in g:
            ok &= eq(self.h_b_dst, self.w3b, self.ld3b.off["dst"][0])
        if "c5" in g:
            ok &= eq(self.h_res[2:3], self.w5, self.d5)            # the last collective's result (fcollect) is what d5 holds
        if "c1" in g:
            ok &= eq(self.h_A, self.w1, self.A)
        if "c4" in g:
            ok &= eq(self.h_deg, self.w4, self.deg) and eq(self.h_par, self.w4, self.par)
            ok &= bool(torch.equal(self.h_fdeg, self.f_deg.cpu())) and bool(torch.equal(self.h_fpar, self.f_par.cpu()))
        return bool(ok)

    def e2e_step_pipelined(self):
        """Pipelined form: uploads on one stream, library calls on the main stream, read-backs on a third one, chained with
        events, so the upload of segment k + 1 overlaps the read-back of segment k (PCIe is full duplex: 55 + 57 GB/s one
        way at a time, 100 GB/s together on this box).  Hazards: an upload waits for the library call of the previous
        segment (it may overwrite that call's inputs); a library call waits for its own upload and for the read-back of the
        previous segment (it may overwrite what is still being read).  One event pair around each class of segments (copy,
        AMO); returns {class: (start, end)}."""
        torch = self.torch
        main = torch.cuda.current_stream()
        if not hasattr(self, "s_up"):
            self.s_up, self.s_dn = torch.cuda.Stream(), torch.cuda.Stream()
        ev = lambda: torch.cuda.Event()                                       # noqa: E731
        out, segs = {}, self._e2e_segments()
        for cls in ("copy", "amo"):
            mine = [x for x in segs if x[1] == cls]
            if not mine:
                continue
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(main)
            prev_c, prev_d = a, None
            for _name, _cls, up, call, down in mine:
                self.s_up.wait_event(prev_c)
                with torch.cuda.stream(self.s_up):
                    up()
                    u = ev(); u.record(self.s_up)
                main.wait_event(u)
                if prev_d is not None:
                    main.wait_event(prev_d)
                call()
                c = ev(); c.record(main)
                self.s_dn.wait_event(c)
                with torch.cuda.stream(self.s_dn):
                    down()
                    d = ev(); d.record(self.s_dn)
                prev_c, prev_d = c, d
            main.wait_event(prev_d)
            b.record(main)
            out[cls] = (a, b)
        return out

    # ---- verification against the CPU oracle, after the timed loops and outside every timed region ------------------------
    def verify(self, ob):
        """Every segment's library call is made once more on the same inputs and its result buffers are compared with the
        CPU oracle's (`ob`: an OracleBench holding the same inputs): bit-exact for copies, integer atomics and the fp32
        reduction (the oracle accumulates in fp64 in PE order, as the kernel does); fetched values of fetch-add / compare-swap
        through schedule-independent invariants.  Raises AssertionError on the first mismatch; returns {segment: True}."""
        torch, inp, g, ok = self.torch, self.inp, self.inp.groups, {}
        host = lambda t: t.cpu().numpy()                                           # noqa: E731
        if "c3a" in g:
            n, b = inp.c3a_npes, inp.c3a_blk
            self.w3a.view(self.a_dst, n * b).zero_()
            self.w3a.alltoall(self.a_dst, self.a_src, b)
            ob.o3a.alltoall(ob.a_dst, ob.a_src, b)
            assert np.array_equal(host(self.w3a.view(self.a_dst, n * b)), ob.o3a.view(ob.a_dst, n * b)), "alltoall"
            ok["alltoall"] = True
        if "c3b" in g:
            ob.o3b.exec_ops(ob.ops3b)
            want = ob.o3b.obj("dst")
            for name, run in (("put_batch_skewed", lambda: self.w3b.enqueue_batch(self.b3b)),
                              ("put_batch_skewed_onecall", lambda: self.w3b.enqueue_batch_dev(
                                  self.ops3b_dev, self.plan_us["put_batch_skewed"]["nops"], self.work3b))):
                self.ld3b.obj("dst").zero_()
                run()
                assert np.array_equal(host(self.ld3b.obj("dst")), want), name
                ok[name] = True
            assert self.w3b.batch_status(self.work3b) == (0, 0)
        if "c5" in g:
            n, nb = inp.c5_npes, inp.c5_bytes
            for name, gpu, orc_ in (
                    ("sum_reduce_f32", lambda: self.w5.sum_reduce(0, self.d5, self.s_f32, nb // 4),
                     lambda: ob.o5.sum_reduce_f32(ob.d5, ob.s_f32, nb // 4)),
                    ("sum_reduce_i64", lambda: self.w5.sum_reduce(1, self.d5, self.s_i64, nb // 8),
                     lambda: ob.o5.sum_reduce_i64(ob.d5, ob.s_i64, nb // 8)),
                    ("fcollect", lambda: self.w5.fcollect(self.d5, self.s_fc, inp.c5_fc_bytes),
                     lambda: ob.o5.fcollect(ob.d5, ob.s_fc, inp.c5_fc_bytes))):
                self.w5.view(self.d5, nb).zero_()
                ob.o5.view(ob.d5, nb)[:] = 0
                gpu(); orc_()
                assert np.array_equal(host(self.w5.view(self.d5, nb)), ob.o5.view(ob.d5, nb)), name
                ok[name] = True
        if "c1" in g:
            c = inp.c1
            self.w1.view(self.A, c.nelem * 8).zero_()
            e0 = self.w1.barrier_epoch()
            self.w1.atomic_add_batch(self.A, self.c1_t, self.c1_i, val=self.c1_v, flags=self.flags | self.c1_flags)
            assert self.w1.barrier_epoch() == e0 + 1, "the folded barrier did not happen"
            ob.o1.view(ob.A, c.nelem * 8)[:] = 0
            ob.o1.atomic_add_batch(ob.A, c.tgt_pe, c.idx, c.val)
            assert np.array_equal(host(self.w1.view(self.A, c.nelem * 8)), ob.o1.view(ob.A, c.nelem * 8)), "atomic_add"
            ok["atomic_add"] = True
        if "c4" in g:
            q, vpp = inp.c4, inp.c4.verts_per_pe
            self.w4.view(self.deg, vpp * 8).zero_()
            self.w4.view(self.par, vpp * 8).fill_(255)
            self.w4.atomic_fetch_add_batch(self.deg, self.c4_ou, self.c4_lu, self.f_deg, val=None, val_scalar=1, flags=self.fadd_flags)
            self.w4.atomic_compare_swap_batch(self.par, self.c4_ov, self.c4_lv, self.f_par, cond=None, cond_scalar=M64,
                                              val=self.c4_val, flags=self.cas_flags)
            ob.o4.view(ob.deg, vpp * 8)[:] = 0
            ou, lu, ov, lv, ones, cond, val = ob.c4
            ob.o4.atomic_fetch_add_batch(ob.deg, ou, lu, ones)
            deg = host(self.w4.view(self.deg, vpp * 8, torch.int64)).reshape(-1)
            assert ob.nedge == len(q.u) and np.array_equal(deg, ob.o4.view(ob.deg, vpp * 8, np.int64).reshape(-1)), "degrees"
            # fetch-add(1): the fetched values of a word are a permutation of 0 .. k-1.  Complete check in O(E): every op is
            # sent to slot start[word] + fetched (start = exclusive prefix sum of the exact degrees, so the slots of a word are
            # its own k consecutive ones once the range check has passed); E ops into E slots hit every slot iff no two ops of
            # a word fetched the same value.
            from paper_2607_08006_b200.binding import AMO_HOT_AGGREGATE
            if self.fadd_flags & AMO_HOT_AGGREGATE:
                assert self.w4.amo_last_path() == 1, "fetch-add: the hot-set kernels did not run (plain kernel timed instead)"
            f = host(self.f_deg)
            k = deg.astype(np.int64)
            assert int(k.sum()) == len(f) and (f >= 0).all() and (f < k[q.u]).all(), "fetched degree out of range"
            seen = np.zeros(len(f), dtype=bool)
            seen[(np.cumsum(k) - k)[q.u] + f] = True
            assert seen.all(), "fetch-add: the fetched values of a word are not a permutation of 0 .. k-1"
            del seen
            # compare-swap(-1 -> u): one winner per touched slot, the slot holds the winner's u (an in-neighbour of v by
            # construction: u is the source of the very edge whose op won), every loser fetched the final value
            par = host(self.w4.view(self.par, vpp * 8, torch.int64)).reshape(-1)
            fp = host(self.f_par)
            won = fp == -1
            assert np.array_equal(np.bincount(q.v[won], minlength=len(par)), (np.bincount(q.v, minlength=len(par)) > 0).astype(np.int64)), "slot not claimed exactly once"
            assert np.array_equal(par[q.v[won]], q.u[won].astype(np.int64)), "parent is not the winner's source vertex"
            assert np.array_equal(fp[~won], par[q.v[~won]]), "a losing compare-swap fetched something else than the final parent"
            assert (par[np.bincount(q.v, minlength=len(par)) == 0] == -1).all(), "untouched parent slot modified"
            ok["atomic_fetch_add"] = ok["atomic_compare_swap"] = True
        if "next4" in g:
            t = inp.fft
            block, nblocks, sbs, sps, dbs, dps = t.params()
            self.wf.view(self.f_dst, t.slab_bytes).zero_()
            self.wf.alltoalls(self.f_dst, self.f_src, dps, sps, dbs, sbs, block, nblocks)
            ow = ob.orc.OracleWorld(t.npes, 2 * t.slab_bytes + 512)
            os_, od = ow.malloc(t.slab_bytes), ow.malloc(t.slab_bytes)
            ow.view(os_, t.slab_bytes)[:] = t.A
            ow.alltoalls(od, os_, dps, sps, dbs, sbs, block, nblocks)
            assert np.array_equal(host(self.wf.view(self.f_dst, t.slab_bytes)), ow.view(od, t.slab_bytes)), "fft transpose"
            ok["next4_fft_transpose_alltoalls"] = True
            n, b = inp.sh_npes, inp.sh_blk
            for ws in self.wsh:
                ws.view(self.sh_dst, n * b).zero_()
            for ws in self.wsh:
                ws.galltoall(self.sh_dst, self.sh_src, b)
            ow = ob.orc.OracleWorld(n, 2 * n * b + 512)                  # the GLOBAL world of all the PEs
            os_, od = ow.malloc(n * b), ow.malloc(n * b)
            ow.view(os_, n * b)[:] = inp.sh_payload
            ow.alltoall(od, os_, b)
            for sh, ws in enumerate(self.wsh):
                assert np.array_equal(host(ws.view(self.sh_dst, n * b)), ob.orc.shard_rows(ow, sh, 2, od, n * b)), "sharded alltoall"
            ok["next4_sharded_alltoall_2_shards_on_one_gpu"] = True
        if "c2" in g:
            h, w, fb = inp.halo, self.w2, inp.halo.face_bytes
            send_off = self.ld2.off["send"][0]
            self.ld2.obj("sig").zero_()
            self.ld2.obj("ghost").zero_()
            snaps = {}
            for r in range(1, HALO_ROUNDS + 1):                      # the 50 rounds of the timed step once more
                w.app_halo_perturb(self.U_off, h.B, h.seed, r)
                w.app_halo_pack(send_off, self.U_off, h.B)
                if r > HALO_ROUNDS - 2:
                    snaps[r] = host(self.ld2.obj("send")).copy()     # what the last two rounds send (one per ghost parity)
                w.enqueue_batch(self.halo_batches[r - 1])
            ghost, sig = host(self.ld2.obj("ghost")), host(self.ld2.obj("sig"))
            o2 = ob.o2
            o2.obj("ghost")[:] = 0
            o2.obj("sig")[:] = 0
            for r in sorted(snaps):
                o2.obj("send")[:] = snaps[r]
                o2.exec_ops(ob.ops2[r - 1])
            assert np.array_equal(ghost, o2.obj("ghost")) and np.array_equal(sig, o2.obj("sig")), "halo ghosts / signal words"
            ok["halo_put_signal_wait_event_pairs"] = True
            # the timed form: the 50 rounds replayed from the CUDA graph of the library's launches (every round sends what
            # `send` holds; rounds 49 and 50 fill the two ghost parities, the signal words end at 50)
            if self.halo_graphs is not None:
                self.ld2.obj("ghost").zero_()
                self.ld2.obj("sig").zero_()
                self.halo_graphs[0].replay()
                o2.obj("ghost")[:] = 0
                o2.obj("sig")[:] = 0
                o2.obj("send")[:] = host(self.ld2.obj("send"))
                for r in (HALO_ROUNDS - 1, HALO_ROUNDS):
                    o2.exec_ops(ob.ops2[r - 1])
                assert np.array_equal(host(self.ld2.obj("ghost")), o2.obj("ghost")), "halo ghosts after the graph replay"
                assert np.array_equal(host(self.ld2.obj("sig")), o2.obj("sig")), "halo signal words after the graph replay"
                ok["halo_put_signal_wait"] = True
                self.ld2.obj("ghost").zero_()
                self.ld2.obj("sig").zero_()
                self.halo_graphs[3].replay()
                assert w.batch_status() == (0, 0)
                assert np.array_equal(host(self.ld2.obj("ghost")), o2.obj("ghost")), "halo ghosts after the one-call graph replay"
                assert np.array_equal(host(self.ld2.obj("sig")), o2.obj("sig")), "halo signal words after the one-call graph replay"
                ok["halo_put_signal_wait_onecall_graph"] = True
                o2.obj("ghost")[:] = 0
                o2.obj("sig")[:] = 0
                for r in sorted(snaps):
                    o2.obj("send")[:] = snaps[r]
                    o2.exec_ops(ob.ops2[r - 1])
            self.ld2.obj("ghost").zero_()                            # the same two rounds through the one-call form
            self.ld2.obj("sig").zero_()
            for r in sorted(snaps):
                self.ld2.obj("send").copy_(torch.from_numpy(snaps[r]))
                w.enqueue_batch_dev(self.halo_ops_dev[r - 1], 96)
            assert w.batch_status() == (0, 0)
            assert np.array_equal(host(self.ld2.obj("ghost")), o2.obj("ghost")) and np.array_equal(host(self.ld2.obj("sig")), o2.obj("sig")), "halo, one-call form"
            ok["halo_put_signal_wait_onecall"] = True
        return ok

    # ---- ceilings measured in the same run ---------------------------------------------------------------------------
    def back_to_back(self, nrep=4, reps=3):
        """The single-launch copy-class segments once more, each as a CUDA graph of `nrep` back-to-back launches inside ONE
        event pair (every launch streams 0.4 - 1 GB, far more than the 126 MB L2, so nothing is reused between launches):
        microseconds per launch without the 6 us an event pair adds around a single launch.  Reported beside the per-launch
        event-pair figures, not part of `value`."""
        torch, inp, g, calls = self.torch, self.inp, self.inp.groups, {}
        if "c3a" in g:
            calls["alltoall"] = lambda: self.w3a.alltoall(self.a_dst, self.a_src, inp.c3a_blk)
        if "c3b" in g:
            calls["put_batch_skewed"] = lambda: self.w3b.enqueue_batch(self.b3b)
        if "c5" in g:
            n = inp.c5_bytes
            calls["sum_reduce_f32"] = lambda: self.w5.sum_reduce(0, self.d5, self.s_f32, n // 4)
            calls["sum_reduce_i64"] = lambda: self.w5.sum_reduce(1, self.d5, self.s_i64, n // 8)
            calls["fcollect"] = lambda: self.w5.fcollect(self.d5, self.s_fc, inp.c5_fc_bytes)
        out = {}
        for name, fn in calls.items():
            fn()
            torch.cuda.synchronize()
            gr = torch.cuda.CUDAGraph()
            with torch.cuda.graph(gr, capture_error_mode="thread_local"):
                for _ in range(nrep):
                    fn()
            ts = []
            for _ in range(reps + 1):
                a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                a.record(); gr.replay(); b.record(); b.synchronize()
                ts.append(a.elapsed_time(b) * 1e3 / nrep)
            out[name] = statistics.mean(ts[1:])
        return out

    def ceilings(self, reps=5):
        """L2-atomic ceilings (bare red / atom / cas at hashed addresses, include/shmemg_probe.h) on the C1 and C4
        footprints, and the library's own plain-copy rate on the C5 world.  Returns Mops/s and GB/s (best of reps)."""
        torch, inp, g = self.torch, self.inp, self.inp.groups
        out = {}

        def best(fn, units):
            ts = []
            for _ in range(reps + 1):
                a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                a.record(); fn(); b.record(); b.synchronize()
                ts.append(a.elapsed_time(b))
            return units / (min(ts[1:]) * 1e-3)
        if "c1" in g:
            n = 1 << 24
            out["red_add_512KiB_Mops"] = best(lambda: self.w1.probe_atomic(0, self.A, inp.c1.nelem, n), n) / 1e6
            # (iv) ONE address, without / with warp aggregation
            out["red_add_single_address_Mops"] = best(lambda: self.w1.probe_atomic_stream(0, self.A, None, None, n), n) / 1e6
            out["red_add_single_address_warp_aggregated_Mops"] = best(lambda: self.w1.probe_atomic_stream(0, self.A, None, None, n, True), n) / 1e6
            out["atom_add_single_address_Mops"] = best(lambda: self.w1.probe_atomic_stream(1, self.A, None, None, n >> 2), n >> 2) / 1e6
            out["atom_add_single_address_warp_aggregated_Mops"] = best(lambda: self.w1.probe_atomic_stream(1, self.A, None, None, n, True), n) / 1e6
            # what an event pair around the smallest possible kernel costs in this run (launch floor of a 65 536-op batch)
            out["empty_kernel_event_pair_us"] = 1e6 / best(lambda: self.w1.barrier_all(), 1)
        if "c4" in g:
            n, vpp = len(inp.c4.u), inp.c4.verts_per_pe
            out["red_add_32MiB_Mops"] = best(lambda: self.w4.probe_atomic(0, self.deg, vpp, n), n) / 1e6
            out["atom_add_32MiB_Mops"] = best(lambda: self.w4.probe_atomic(1, self.deg, vpp, n), n) / 1e6
            out["atom_cas_32MiB_Mops"] = best(lambda: self.w4.probe_atomic(2, self.par, vpp, n), n) / 1e6
            # (iii) the bare atomic on the RMAT address stream itself (operands read, nothing written), without / with warp aggregation
            for nm, mode, t_, i_, off in (("atom_add", 1, self.c4_ou, self.c4_lu, self.deg), ("red_add", 0, self.c4_ou, self.c4_lu, self.deg),
                                          ("atom_cas", 2, self.c4_ov, self.c4_lv, self.par)):
                out[nm + "_rmat_stream_Mops"] = best(lambda: self.w4.probe_atomic_stream(mode, off, t_, i_, n), n) / 1e6
                out[nm + "_rmat_stream_warp_aggregated_Mops"] = best(lambda: self.w4.probe_atomic_stream(mode, off, t_, i_, n, True), n) / 1e6
        if "c5" in g:
            nb = inp.c5_bytes
            out["copy_all_GBps"] = best(lambda: self.w5.probe_copy_all(self.d5, self.s_f32, nb), 2 * inp.c5_npes * nb) / 1e9
        return out


# ======================================================================================================================
# oracle arm: the CPU oracle as it stands (single thread), on a bounded sample of the same step
# ======================================================================================================================
class OracleBench:
    """Bounded sample of one step (defaults: the whole step except the barrier-latency loops and the halo application
    compute, about 5-10 s on one core): C3a and C3b whole; C2 `halo_rounds` exchange rounds; C5 sum_reduce on the first
    1/`reduce_div` of the elements (all PEs), fcollect whole; C1 whole; C4 the first 2^`c4_log2` edges."""

    def __init__(self, inp: Inputs, halo_rounds=HALO_ROUNDS, reduce_div=1, c4_log2=26):
        from oracle import oracle as orc
        self.orc, self.inp = orc, inp
        g = inp.groups
        self.halo_rounds, self.reduce_div = halo_rounds, reduce_div
        self.sample = []
        if "c3a" in g:
            n, b = inp.c3a_npes, inp.c3a_blk
            self.o3a = orc.OracleWorld(n, 2 * n * b + 512)
            self.a_src, self.a_dst = self.o3a.malloc(n * b), self.o3a.malloc(n * b)
            self.o3a.view(self.a_src, n * b)[:] = inp.c3a
            self.sample.append("C3a whole")
        if "c3b" in g:
            prog = inp.c3b.prog
            self.o3b = orc.OracleWorld(prog.npes, sum((x + 255) // 256 * 256 for x in prog.obj_bytes) + 512)
            self.o3b.load_program(prog)
            self.ops3b = self.o3b.translate(prog)
            self.sample.append("C3b whole")
        if "c2" in g:
            h = inp.halo
            prog = h.program(with_consume=False, with_U=False)
            self.o2 = orc.OracleWorld(8, sum((x + 255) // 256 * 256 for x in prog.obj_bytes) + 512)
            self.o2.load_program(prog)
            self.o2.obj("send", np.uint64)[:] = np.arange(8 * 6 * h.face_bytes // 8, dtype=np.uint64).reshape(8, -1)
            self.ops2 = [self.o2.translate(h.round_ops(prog, r, False)) for r in range(1, halo_rounds + 1)]
            self.sample.append("C2 %d of %d exchange rounds (library ops only)" % (halo_rounds, HALO_ROUNDS))
        if "c5" in g:
            n, nb = inp.c5_npes, inp.c5_bytes
            self.o5 = orc.OracleWorld(n, 3 * nb + inp.c5_fc_bytes + 1024)
            self.s_f32, self.s_i64, self.d5 = self.o5.malloc(nb), self.o5.malloc(nb), self.o5.malloc(nb)
            self.s_fc = self.o5.malloc(inp.c5_fc_bytes)
            self.o5.view(self.s_f32, nb, np.float32)[:] = inp.c5_f32
            self.o5.view(self.s_i64, nb, np.int64)[:] = inp.c5_i64
            self.o5.view(self.s_fc, inp.c5_fc_bytes)[:] = inp.c5_fc
            self.sample.append("C5 sum_reduce on the first 1/%d of the elements, fcollect whole" % reduce_div)
        if "c1" in g:
            c = inp.c1
            self.o1 = orc.OracleWorld(c.npes, c.nelem * 8 + 512)
            self.A = self.o1.malloc(c.nelem * 8)
            self.sample.append("C1 whole")
        if "c4" in g:
            q = inp.c4
            self.nedge = min(len(q.u), 1 << c4_log2)
            self.o4 = orc.OracleWorld(q.npes, 2 * q.verts_per_pe * 8 + 512)
            self.deg, self.par = self.o4.malloc(q.verts_per_pe * 8), self.o4.malloc(q.verts_per_pe * 8)
            m = self.nedge
            self.c4 = (q.owner(q.u[:m]), q.local(q.u[:m]), q.owner(q.v[:m]), q.local(q.v[:m]),
                       np.ones(m, dtype=np.uint64), np.full(m, M64, dtype=np.uint64), q.u[:m].astype(np.uint64))
            self.sample.append("C4 first %d of %d edges" % (m, len(q.u)))

    def step(self):
        """Returns {segment: (seconds, bytes or ops in the sample)}."""
        inp, g, out = self.inp, self.inp.groups, {}
        tm = time.perf_counter
        if "c3a" in g:
            t = tm(); self.o3a.alltoall(self.a_dst, self.a_src, inp.c3a_blk)
            out["alltoall"] = (tm() - t, 2 * inp.c3a_npes ** 2 * inp.c3a_blk)
        if "c3b" in g:
            t = tm(); self.o3b.exec_ops(self.ops3b)
            out["put_batch_skewed"] = (tm() - t, 2 * int(inp.c3b.sizes.sum()))
        if "c2" in g:
            self.o2.obj("sig")[:] = 0
            t = tm()
            for ops in self.ops2:
                self.o2.exec_ops(ops)
            out["halo_put_signal_wait"] = (tm() - t, self.halo_rounds * 2 * 48 * inp.halo.face_bytes)
        if "c5" in g:
            n, nb, dv = inp.c5_npes, inp.c5_bytes, self.reduce_div
            t = tm(); self.o5.sum_reduce_f32(self.d5, self.s_f32, nb // 4 // dv)
            out["sum_reduce_f32"] = (tm() - t, 2 * n * nb // dv)
            t = tm(); self.o5.sum_reduce_i64(self.d5, self.s_i64, nb // 8 // dv)
            out["sum_reduce_i64"] = (tm() - t, 2 * n * nb // dv)
            t = tm(); self.o5.fcollect(self.d5, self.s_fc, inp.c5_fc_bytes)
            out["fcollect"] = (tm() - t, n * inp.c5_fc_bytes * (n + 1))
        if "c1" in g:
            c = inp.c1
            self.o1.view(self.A, c.nelem * 8)[:] = 0
            t = tm(); self.o1.atomic_add_batch(self.A, c.tgt_pe, c.idx, c.val)
            out["atomic_add"] = (tm() - t, len(c.val))
        if "c4" in g:
            vpp = inp.c4.verts_per_pe
            self.o4.view(self.deg, vpp * 8)[:] = 0
            self.o4.view(self.par, vpp * 8)[:] = 255
            ou, lu, ov, lv, ones, cond, val = self.c4
            t = tm(); self.o4.atomic_fetch_add_batch(self.deg, ou, lu, ones)
            out["atomic_fetch_add"] = (tm() - t, self.nedge)
            t = tm(); self.o4.atomic_compare_swap_batch(self.par, ov, lv, cond, val)
            out["atomic_compare_swap"] = (tm() - t, self.nedge)
        return out


def class_rates(table, seg_seconds, seg_units):
    """(copy GB/s, amo Mops/s) from per-segment seconds and units (bytes for copy-class, ops for amo-class)."""
    cb = sum(seg_units[k] for k in seg_units if table[k]["cls"] == "copy")
    cs = sum(seg_seconds[k] for k in seg_units if table[k]["cls"] == "copy")
    ao = sum(seg_units[k] for k in seg_units if table[k]["cls"] == "amo")
    as_ = sum(seg_seconds[k] for k in seg_units if table[k]["cls"] == "amo")
    return (cb / cs / 1e9 if cs > 0 else 0.0), (ao / as_ / 1e6 if as_ > 0 else 0.0), cs, as_


ALL_GROUPS = ["c1", "c2", "c3a", "c3b", "c4", "c5", "barrier", "next2", "next4"]


def max_over_ranks(dist, device, seg_ms, whole_ms, e2e_ms):
    """Replicas only: every rank runs the same step on its own GPU; a segment's time is the MAX over ranks
    (one all_reduce of a small vector, the only collective of the bench and not on the data path).  Returns
    (names, seg_ms, whole_ms, e2e_ms) with the reduced values; `dist` None = single process."""
    import torch
    names = sorted(seg_ms)
    enames = sorted(e2e_ms) if e2e_ms else []                    # the end-to-end leg has its own keys (segments and pipelined regions)
    vec = torch.tensor([seg_ms[k] for k in names] + [whole_ms] + [e2e_ms[k] for k in enames], dtype=torch.float64, device=device)
    if dist is not None:
        dist.all_reduce(vec, op=dist.ReduceOp.MAX)
    vec = vec.cpu().tolist()
    out_e2e = dict(zip(enames, vec[len(names) + 1:])) if e2e_ms else e2e_ms
    return names, dict(zip(names, vec[:len(names)])), vec[len(names)], out_e2e


def whole_job_units(table, names, steps, world):
    """Units (bytes or ops) all ranks processed in the timed region: weak scaling, every replica does the full step."""
    return {k: table[k].get("bytes", table[k].get("ops")) * steps * world for k in names}


def base_line(args, n_gpus):
    return {"metric": METRIC, "unit": UNIT, "n_gpus": n_gpus, "steps": args.steps, "warmup": args.warmup,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "data": "synthetic",
            "config": {"workload": WORKLOAD + (" [--small development sizes]" if args.small else ""),
                       "parallelism": "replicas only (no sharding, no inter-GPU transport: north_star)",
                       "l2": "inputs larger than L2: one step streams about 4.6 GiB through the 126 MB L2 between two "
                             "uses of any buffer; by-nature L2-resident cases (C1's 512 KiB target, halo faces just packed) "
                             "are kept as the application leaves them",
                       "value_definition": "copy-class algorithmic bytes / summed CUDA-event time of the copy-class "
                                           "segments (library calls only), summed over ranks",
                       "launch": "single collectives and the Zipf batch: one event pair around the one launch; the 50 halo "
                                 "rounds (a launch-bound inner loop, 48 MiB per 10 us launch): replayed from ONE CUDA graph of "
                                 "the 50 pre-planned batch launches, one event pair around the replay; the same launches with "
                                 "an event pair around each are reported as halo_put_signal_wait_event_pairs"}}


def run_reference(args):
    """This tier's reference arm: the oracle, as it stands, on the host cores (rank 0 only)."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    groups = [x for x in (args.only.split(",") if args.only else ALL_GROUPS) if x not in ("barrier", "next4")]
    inp = Inputs(args.small, groups)
    table = segment_table(inp)
    ob = OracleBench(inp)
    for _ in range(min(args.warmup, 1)):
        ob.step()
    secs, units = {}, {}
    t0 = time.perf_counter()
    for _ in range(args.steps):
        for k, (s, u) in ob.step().items():
            secs[k] = secs.get(k, 0.0) + s
            units[k] = units.get(k, 0) + u
    wall = time.perf_counter() - t0
    gbps, mops, _, _ = class_rates(table, secs, units)
    line = base_line(args, args.gpus)
    sample = "; ".join(ob.sample)
    line.update({"impl": "reference", "value": gbps, "amo_mops": mops, "ms_per_step": wall / args.steps * 1e3, "dtype": "u8",
                 "segments": {k: {"ms": secs[k] / args.steps * 1e3,
                                  ("GBps" if table[k]["cls"] == "copy" else "Mops"):
                                      units[k] / secs[k] / (1e9 if table[k]["cls"] == "copy" else 1e6)} for k in secs},
                 "cpu_baseline": {"value": gbps, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
                 "e2e": {"value": gbps, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
                 "gpu_launches": 0})
    print(json.dumps(line))


def run_cuda(args):
    import torch
    rank, world = int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the shmemg hot path has no CPU fallback")
    # SHMEMG_BENCH_ONE_GPU=1 (development only, marked in the JSON line): every rank uses cuda:0 and the rendezvous runs over
    # gloo -- the N > 1 code path on a box with one GPU (NCCL refuses two ranks on one device)
    one_gpu = os.environ.get("SHMEMG_BENCH_ONE_GPU") == "1"
    if one_gpu:
        local = 0
    torch.cuda.set_device(local)
    device = torch.device("cuda", local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        if one_gpu:
            dist.init_process_group("gloo")
        else:
            dist.init_process_group("nccl", device_id=device)
    groups = args.only.split(",") if args.only else ALL_GROUPS
    inp = Inputs(args.small, groups)
    table = segment_table(inp)
    cb = CudaBench(inp, device)

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize(device)

    # ---- device-resident leg ------------------------------------------------------------------------------------------
    for _ in range(args.warmup):
        cb.step()
    barrier()
    sampler = ClockSampler(local)
    sampler.start()
    l0 = cb.launches()
    cb.rec.on = True
    t_a, t_b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t_a.record()
    for _ in range(args.steps):
        cb.step()
    t_b.record()
    barrier()
    clocks = sampler.stop()
    cb.rec.on = False
    launches = cb.launches() - l0
    whole_ms = t_a.elapsed_time(t_b)
    seg_ms = cb.rec.totals_ms()                                   # summed over the K steps
    cb.rec.pairs = []

    # ---- end-to-end leg ---------------------------------------------------------------------------------------------------
    e2e_ms, h2d, d2h, e2e_check = None, 0, 0, None
    if not args.no_e2e:
        cb.setup_e2e()
        cb.e2e_step()
        barrier()
        cb.h2d = cb.d2h = 0
        cb.rec.on = True
        for _ in range(args.steps):
            cb.e2e_step()
        barrier()
        cb.rec.on = False
        e2e_ms = cb.rec.totals_ms()
        h2d, d2h = cb.h2d // args.steps, cb.d2h // args.steps
        cb.rec.pairs = []
        # the same transfers and calls, pipelined over three streams (upload / call / read-back)
        cb.e2e_step_pipelined()
        barrier()
        regions = [cb.e2e_step_pipelined() for _ in range(args.steps)]
        barrier()
        for cls in ("copy", "amo"):
            if regions and cls in regions[0]:
                e2e_ms["__pipelined_" + cls] = sum(r[cls][0].elapsed_time(r[cls][1]) for r in regions)
        e2e_check = cb.e2e_check()
    ceil = cb.ceilings() if rank == 0 else {}
    b2b = cb.back_to_back() if rank == 0 else {}

    # ---- max over ranks of every segment time ---------------------------------------------------------------------------
    names, seg_ms, whole_ms, e2e_ms = max_over_ranks(dist, device, seg_ms, whole_ms, e2e_ms)
    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    K = args.steps
    units = whole_job_units(table, names, K, world)
    secs = {k: seg_ms[k] * 1e-3 for k in names}
    gbps, mops, copy_s, amo_s = class_rates(table, secs, units)
    peak, peak_src = measured_peaks()
    segments = {}
    for k in names:
        t, per_launch_ms = table[k], seg_ms[k] / (K * table[k]["launches"])
        d = {"kernel": t["kernel"], "ms_per_step": seg_ms[k] / K, "launches_per_step": t["launches"]}
        if t["cls"] == "copy":
            d["GBps"] = units[k] / world / secs[k] / 1e9
            d["frac_of_measured_hbm"] = d["GBps"] / peak
            d["frac_of_nominal_8TBps"] = d["GBps"] / 8000.0
        elif t["cls"] == "amo":
            d["Mops"] = units[k] / world / secs[k] / 1e6
        elif t["cls"] == "xcopy":
            d["GBps"] = units[k] / world / secs[k] / 1e9
            d["frac_of_measured_hbm"] = d["GBps"] / peak
            d["in_headline"] = False
        elif t["cls"] == "xtime":
            d["us_per_round"] = seg_ms[k] / K / t["ops"] * 1e3
            d["in_headline"] = False
        elif t["cls"] == "xamo":
            d["Mops"] = units[k] / world / secs[k] / 1e6
            d["in_headline"] = False
            if "bytes_per_op" in t:
                d["bytes_per_op"] = t["bytes_per_op"]
                d["frac_of_measured_hbm"] = d["Mops"] * 1e6 * t["bytes_per_op"] / 1e9 / peak
        else:
            d["us_per_barrier"] = seg_ms[k] / K / t["ops"] * 1e3
        d["us_per_launch"] = per_launch_ms * 1e3
        if k in b2b:                                              # the same launch back to back from a CUDA graph (rank 0)
            d["back_to_back_us_per_launch"] = b2b[k]
            d["back_to_back_GBps"] = t["bytes"] / t["launches"] / b2b[k] / 1e3
            d["back_to_back_frac_of_measured_hbm"] = d["back_to_back_GBps"] / peak
        if k in cb.plan_us:
            d["host_planning"] = dict(cb.plan_us[k], note="shmemg_batch_plan_bytes + shmemg_batch_create per batch (host pass, H2D, "
                                      "stream sync); done once before the timed region, the plan is re-enqueued every step "
                                      "(plan_reused: true); the one-call segment beside this one plans on the device inside "
                                      "the timed region", plan_reused=True)
        if t["cls"] == "amo" and "bytes_per_op" in t:
            d["bytes_per_op"] = t["bytes_per_op"]
            d["operand_stream_GBps"] = d["Mops"] * 1e6 * t["bytes_per_op"] / 1e9
            d["frac_of_measured_hbm"] = d["operand_stream_GBps"] / peak
        segments[k] = d
    if "atomic_add" in segments and "red_add_512KiB_Mops" in ceil:
        segments["atomic_add"]["frac_of_l2_atomic_ceiling"] = segments["atomic_add"]["Mops"] / ceil["red_add_512KiB_Mops"]
    if "atomic_fetch_add" in segments and "atom_add_32MiB_Mops" in ceil:
        segments["atomic_fetch_add"]["frac_of_l2_atomic_ceiling"] = segments["atomic_fetch_add"]["Mops"] / ceil["atom_add_32MiB_Mops"]
    if "atomic_fetch_add" in segments and "atom_add_rmat_stream_Mops" in ceil:
        segments["atomic_fetch_add"]["vs_bare_atom_add_on_the_same_stream"] = segments["atomic_fetch_add"]["Mops"] / ceil["atom_add_rmat_stream_Mops"]
    if "atomic_compare_swap" in segments:
        segments["atomic_compare_swap"]["note"] = ("test-before-swap: most of the 2^26 ops are resolved by a load (served by L1 for the hot "
                                                   "slots), so the atom.cas probe does not bound this variant; its HBM traffic is the operand / "
                                                   "result stream (bytes_per_op, frac_of_measured_hbm) plus one 32-byte sector per slot that is "
                                                   "claimed; the random 8-byte test loads are L2 hits (32 MiB of slots)")
    if "atomic_compare_swap_plain" in segments and "atom_cas_32MiB_Mops" in ceil:
        segments["atomic_compare_swap_plain"]["frac_of_l2_atomic_ceiling"] = segments["atomic_compare_swap_plain"]["Mops"] / ceil["atom_cas_32MiB_Mops"]
        if "atom_cas_rmat_stream_Mops" in ceil:
            segments["atomic_compare_swap_plain"]["vs_bare_atom_cas_on_the_same_stream"] = segments["atomic_compare_swap_plain"]["Mops"] / ceil["atom_cas_rmat_stream_Mops"]
    if "atomic_add_steady_2p24" in segments and "red_add_512KiB_Mops" in ceil:
        segments["atomic_add_steady_2p24"]["frac_of_l2_atomic_ceiling"] = segments["atomic_add_steady_2p24"]["Mops"] / ceil["red_add_512KiB_Mops"]
    if "atomic_add" in segments and "empty_kernel_event_pair_us" in ceil:
        segments["atomic_add"]["empty_kernel_event_pair_us"] = ceil["empty_kernel_event_pair_us"]

    # dominant copy-class kernel = largest share of the timed copy-class step time
    roofline = None
    copy_names = [k for k in names if table[k]["cls"] == "copy"]
    traffic = ncu_traffic()
    if copy_names:
        by_kernel = {}
        for k in copy_names:
            e = by_kernel.setdefault(table[k]["kernel"], [0.0, 0, 0, 0, True])
            e[0] += secs[k]; e[1] += units[k] // world; e[2] += table[k]["launches"] * K
            e[3] += traffic.get(k, 0) * table[k]["launches"] * K
            e[4] = e[4] and k in traffic
        kern = max(by_kernel, key=lambda x: by_kernel[x][0])
        s_all = by_kernel[kern][0]

        def launch_kind(sel):
            """bytes, seconds, launches and ncu DRAM traffic of the dominant kernel's segments picked by `sel`"""
            ks = [k for k in copy_names if table[k]["kernel"] == kern and sel(table[k])]
            if not ks:
                return None
            b = sum(units[k] // world for k in ks); s = sum(secs[k] for k in ks); nl = sum(table[k]["launches"] * K for k in ks)
            tr_ok = all(k in traffic for k in ks) and not inp.small
            tr = sum(traffic.get(k, 0) * table[k]["launches"] * K for k in ks)
            return {"segments": ks, "achieved": b / s / 1e9, "algorithmic_bytes_per_launch": b // nl, "avg_launch_us": s / nl * 1e6,
                    "traffic": (tr // nl) if tr_ok else None}
        hbm_kind = launch_kind(lambda t: not t.get("l2_resident"))
        l2_kind = launch_kind(lambda t: bool(t.get("l2_resident")))
        head = hbm_kind or l2_kind
        # the HBM fraction is quoted for the kernel's HBM-bound launches only; its L2-resident launches (the halo rounds, whose
        # 72 MiB of faces and ghost layers never leave the 126 MB L2: DRAM traffic 0.5x the algorithmic bytes) are listed beside
        # it WITHOUT a fraction: no independent L2 -> SM -> L2 copy ceiling has been measured on this box
        roofline = {"bound": "hbm", "kernel": kern, "achieved": head["achieved"], "peak": peak, "unit": "GB/s",
                    "frac": head["achieved"] / peak, "peak_source": peak_src, "share_of_copy_time": s_all / copy_s,
                    "launches_counted": head["segments"],
                    "algorithmic_bytes_per_launch": head["algorithmic_bytes_per_launch"], "avg_launch_us": head["avg_launch_us"],
                    "traffic": head["traffic"],
                    "traffic_source": "profiles/%s (ncu --set full capture; launch-weighted mean over the counted segments)" % TRAFFIC_CSV,
                    "note": "k_batch_exec runs the Zipf put batch (HBM-bound: 392 MB per launch) and the 50 halo rounds (L2-resident). "
                            "`achieved`, `frac` and `traffic` are those of the HBM-bound launches only (one launch timed by an event "
                            "pair; `segments.put_batch_skewed.back_to_back_*` is the same launch four times from a graph); the halo "
                            "launches are under `l2_resident_launches` and are bound by launch + completion latency and the SMs' own "
                            "L2 ports (profiles/r02b_halo_graph.md), not by HBM"}
        if hbm_kind and l2_kind:
            roofline["l2_resident_launches"] = dict(l2_kind, peak=None, frac=None, unit="GB/s",
                                                    note="L2 traffic rate, not an HBM figure; no measured L2 copy ceiling to divide by")

    line = base_line(args, world)
    if one_gpu:
        line["config"]["workload"] += " [SHMEMG_BENCH_ONE_GPU: all ranks share cuda:0, development only]"
    # the copy class split by where its bytes live: HBM-bound segments (alltoall, Zipf batch, reductions, fcollect) against the
    # measured HBM copy peak; the L2-resident halo rounds on their own (an L2 rate: no HBM fraction is claimed for it)
    def _rate(ks):
        return (sum(units[k] for k in ks) / sum(secs[k] for k in ks) / 1e9) if ks else None
    hbm_ks = [k for k in copy_names if not table[k].get("l2_resident")]
    l2_ks = [k for k in copy_names if table[k].get("l2_resident")]
    class_split = {"hbm_GBps": _rate(hbm_ks), "hbm_frac_of_measured_peak": (_rate(hbm_ks) / peak / world) if hbm_ks else None,
                   "hbm_segments": hbm_ks, "l2_resident_GBps": _rate(l2_ks), "l2_resident_segments": l2_ks}
    line.update({"copy_class_split": class_split})
    line.update({"value": gbps, "amo_mops": mops, "ms_per_step": whole_ms / K,
                 "timed_ms_per_step": sum(v for k, v in seg_ms.items() if table[k]["cls"] != "xtime") / K, "dtype": "u8 (copies), u64 (AMOs), f64-accumulated f32 / i64 (sum_reduce)",
                 "segments": segments, "ceilings": ceil, "roofline": roofline, "clocks": clocks, "gpu_launches": launches,
                 "input_generation_s": inp.gen_seconds})
    if e2e_ms:
        eu = {k: units[k] for k in names if k in e2e_ms and table[k]["cls"] != "sync"}
        es = {k: e2e_ms[k] * 1e-3 for k in eu}
        eg_serial, em_serial, _, _ = class_rates(table, es, eu)
        eg, em = eg_serial, em_serial
        pc, pa = e2e_ms.get("__pipelined_copy"), e2e_ms.get("__pipelined_amo")
        if pc:                                                   # the same bytes / ops over the pipelined regions' times
            eg = sum(v for k, v in eu.items() if table[k]["cls"] == "copy") / (pc * 1e-3) / 1e9
        if pa:
            em = sum(v for k, v in eu.items() if table[k]["cls"] == "amo") / (pa * 1e-3) / 1e6
        line["e2e"] = {"value": eg, "unit": UNIT, "amo_mops": em, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                       "ms_per_step": ((pc or 0.0) + (pa or 0.0)) / K if (pc or pa) else sum(es.values()) / K * 1e3,
                       "serial": {"value": eg_serial, "amo_mops": em_serial, "ms_per_step": sum(es.values()) / K * 1e3},
                       "results_read_back_equal_the_device_results": e2e_check,
                       "note": "every step copies every input from pinned host memory and reads every result back to pinned host "
                               "memory inside the timed region; `value` pipelines the segments over three streams (upload / library "
                               "call / read-back, so the upload of one segment overlaps the read-back of the previous one: PCIe is "
                               "full duplex), one event pair around each class of segments; `serial` runs upload, call and read-back "
                               "of every segment on one stream inside its own event pair; the two batch workloads use the one-call "
                               "form: their descriptors are copied from pinned host memory and planned on the device inside the "
                               "timed region (no plan is reused)"}
    if world == 1 and not args.no_cpu:
        ob = OracleBench(inp)
        res = ob.step()
        if not args.no_verify:                                    # the oracle is test infrastructure: only here and in cpu_baseline
            line["verified"] = cb.verify(ob)
            for k, v in line["verified"].items():
                if k in segments:
                    segments[k]["verified"] = v
        osecs = {k: v[0] for k, v in res.items()}
        ounits = {k: v[1] for k, v in res.items()}
        og, om, ocs, oas = class_rates(table, osecs, ounits)
        line["cpu_baseline"] = {"value": og, "unit": UNIT, "amo_mops": om, "cores": 1, "kind": "oracle",
                                "sample": "; ".join(ob.sample), "seconds": sum(osecs.values()),
                                "host_cores_available": os.cpu_count()}
    print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()


def main():
    args = parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_cuda(args)


if __name__ == "__main__":
    main()
