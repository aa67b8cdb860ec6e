// batch_plan.cuh -- the PLAN FORMAT shared by the host planner (batch.cu), the device planner (plan_dev.cu) and the batch
// executor kernel (batch.cu): 64-byte self-contained tile records in batch order, 64-byte AMO / wait records, completion
// counters.  Not part of the public boundary; shares nothing with oracle/.
#pragma once
#include <stddef.h>

#include "internal.cuh"

#define EXEC_THREADS 192          // warp 0: loader, warp 1: storer, warps 2-5: generic
#define GEN_THREADS 128
#define GEN_FIRST 64
#define GEN_SLOTS 2
#define GEN_TILE 16384u           // bytes per register-path copy tile
#define AMO_RUN_MAX GEN_THREADS
#define TMA_MIN_SPLIT 2048u       // below this, a transfer with unaligned ends is one register-path tile
#define SEG_TILES_MAX 8u          // planner tiles (SHMEMG_TMA_TILE) per segment (256 KiB)
// Executor ring geometry, chosen per batch by the planner (measured on B200, profiles/r01c):
//   latency-bound batches (about one segment per SM): 12 stages of 16 KiB -- small stages start the store front early
//     and a <= 192 KiB segment is loaded without re-using a stage (halo round 16.5 -> 15.1 us);
//   streaming batches: 7 stages of 32 KiB -- 224 KiB in flight per SM towards HBM (C3b 72.6 -> 69.5 us).
#define EXEC_STAGES_MAX 12
#define EXEC_SMEM_MAX (7u * 32768u)
#define EXEC_SMALL_PER_SM (256u * 1024u)   // bulk bytes per SM at or below which a batch counts as latency-bound
#define TRACE_SLOTS 8
#define TRACE_CTAS 256
#define TRACE_BYTES (TRACE_CTAS * TRACE_SLOTS * 8)   // per-CTA timestamps (SHMEMG_TRACE=1)
#define PLAN_CHUNK_OPS 512u       // a run of AMOs / waits never crosses a multiple of this op index (the device planner's chunk)
#define WAIT_RUN_MAX GEN_THREADS  // consecutive waits (of any PEs) polled by one tile, one per generic thread

// tile kinds (bits 0-7 of TileRec.kind); bits 8-15 hold sig_op (put_signal)
enum { T_TMA = 1, T_COPY = 2, T_AMO = 3, T_WAIT = 4, T_NODATA = 5, T_END = 6 };
#define TF_SEGEND 0x00010000u     // (ring only) last bulk tile of its segment: account when its store has completed
#define TF_SIGNAL 0x00020000u     // op is a PUT_SIGNAL
#define TF_CNT_PE 0x00040000u     // a later marker of this PE depends on this op: bump done[initiator]
#define TF_CNT_ALL 0x00080000u    // a later BARRIER_ALL depends on this op: bump done[npes]
#define TF_DEPS 0x00100000u       // dep_pe / dep_all are non-zero
#define TF_ACCT (TF_SIGNAL | TF_CNT_PE | TF_CNT_ALL)

struct TileRec {          // 64 B, self-contained
    uint64_t dst;         // copy destination
    uint64_t src;         // copy source; AMO run / wait run: address of the first AuxRec
    uint64_t sig;         // put_signal: signal word on the target
    uint64_t value;       // signal value
    uint32_t nbytes;      // bytes of this piece (a segment spans several bulk tiles); AMO / wait run: number of records
    uint32_t kind;
    uint32_t op;          // unit index (arrive[op])
    uint32_t nt;          // pieces of this op (arrive[op] advances by nt per launch)
    uint32_t initiator;
    uint32_t dep_pe;      // start when done[initiator] has advanced by dep_pe in this launch
    uint32_t dep_all;     // and done[npes] by dep_all
    uint32_t pe_total;    // how far done[initiator] advances per launch (base of this launch = epoch * pe_total)
};
static_assert(sizeof(TileRec) == 64, "TileRec must be 64 bytes");

struct AuxRec {           // 64 B: one AMO descriptor or one wait condition, resolved on the host
    uint64_t word;        // AMO target word / signal word to poll
    uint64_t fetch;       // AMO fetch slot (0 = none)
    uint64_t value;       // AMO operand / wait comparand
    uint64_t cond;
    uint32_t kind;        // bits 0-7 opcode, bits 8-15 cmp (wait), TF_CNT_*
    uint32_t initiator;
    uint32_t dep_pe;
    uint32_t dep_all;
    uint32_t pe_total;
    uint32_t pad[3];
};
static_assert(sizeof(AuxRec) == 64, "AuxRec must be 64 bytes");

// All run-time counters are MONOTONIC across launches, so a plan needs no re-arming and no exit protocol: one launch
// performs exactly `ntiles` ticket claims, advances done[p] by pe_total[p], done[npes] by all_total and arrive[op] by
// nt; the launch index (epoch) is ticket / ntiles at kernel entry and every threshold is taken relative to it
// (wrap-safe 32-bit differences).
struct PlanHeader {       // 256 B at the start of the plan buffer
    uint32_t ntiles, nunits, npes, trace_on;
    unsigned long long ticket;
    uint32_t all_total, pad1;
    uint64_t tiles_off, aux_off, done_off, arrive_off, trace_off;
    uint64_t pad_a;
    // written by the DEVICE planner (plan_dev.cu) and read by the executor of a one-call batch (shmemg_enqueue_batch);
    // the four words at byte 80 are read with one 16-byte load
    uint32_t stage_bytes, nstages;     // ring geometry
    int32_t status;                    // SHMEMG_OK or the error of the first bad descriptor / SHMEMG_ERR_NOMEM (plan does not fit)
    uint32_t pad2;
    unsigned long long bad_index;      // index of that descriptor
    uint64_t pad3[19];
};
static_assert(sizeof(PlanHeader) == 256, "PlanHeader must be 256 bytes");
static_assert(offsetof(PlanHeader, stage_bytes) == 80, "16-byte aligned geometry words");

// Everything a CTA needs to start is a kernel ARGUMENT (constant bank); the only global reads on the start-up path are
// the first tile record and the ticket counter, issued together.  One-call batches (device planner): `hdr` is set and
// ntiles / all_total / ring geometry are read from the header the planning kernel has just written; the counters of such a
// plan start at zero in every call, so the launch index is 0 and the ticket is not read.
struct ExecArgs {
    const TileRec *tiles;
    unsigned long long *ticket;
    unsigned *done, *arrive;
    unsigned long long *trace;     // nullptr unless SHMEMG_TRACE
    unsigned ntiles, npes, all_total;
    unsigned stage_bytes, nstages;     // ring geometry
    const PlanHeader *hdr;         // nullptr: host-planned batch (everything above is valid)
};

// host-side helpers shared by batch.cu (host planner) and plan_dev.cu (device planner)
int shmemg_exec_smem_attr(shmemg_world *w);
int shmemg_exec_launch(shmemg_world *w, const ExecArgs &a, unsigned grid, size_t smem, cudaStream_t st, bool after_planner);
