// batch.cu -- op-batch planner (host) and the persistent batch executor kernel (sm_100a), plus the single
// put/get/put_signal/wait `_on_stream` calls.  SURVEY.md 8(a) rows a5-a8, a12-a14.
//
// Executor design:
//   * the host planner resolves PE->address translation and cuts every op into self-contained 64-byte TILE RECORDS
//     listed in batch order: bulk-copy tiles (<= 32 KiB, 16-byte aligned), register-path copy tiles (unaligned heads,
//     tails and relatively misaligned transfers), runs of <= 128 AMO descriptors, waits, and no-data tiles;
//   * one CTA per SM, warp-specialised:
//       loader  (1 thread)  claims tiles with a global ticket IN BATCH ORDER, waits for the tile's dependencies,
//                           issues the bulk load (cp.async.bulk global->shared) or hands the tile to the generic
//                           warps;
//       storer  (1 thread)  issues the bulk store (shared->global) when a stage has landed, and when the store has
//                           completed does the tile's completion accounting (arrival, signal, done counters);
//       generic (4 warps)   register-path copies, AMO runs and runs of waits (SIGNAL_WAIT_UNTIL, one per thread).
//     A claimed tile only ever waits for tiles with smaller tickets, which are finished or held by running CTAs whose
//     three roles make progress independently: no deadlock and no co-residency requirement;
//   * ordering state: done[p] = completed ops of PE p, done[npes] = completed ops of all PEs (monotonic, release-
//     incremented).  An op that follows a FENCE/QUIET/WAIT of its PE starts only when done[p] has reached the number
//     of that PE's ops before the marker; an op after a BARRIER_ALL only when done[npes] has reached the number of
//     ops before the barrier (acquire spin).  Only ops that some later op depends on are counted;
//   * the unit of claiming and of completion accounting is the SEGMENT: up to SEG_TILES_MAX consecutive bulk tiles of
//     one op, streamed through one CTA's stage ring; release fences cost microseconds under load, so there is one per
//     segment, not per tile.  An op cut into several pieces completes at its last-ARRIVING piece (acq_rel counter on
//     arrive[op]), which performs the put_signal update with release semantics and the done[] increments.  Ops nobody
//     depends on and that carry no signal do no accounting at all.
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <algorithm>
#include <vector>

#include "tma_stream.cuh"
#include "batch_plan.cuh"

struct shmemg_batch {
    shmemg_world *w;
    uint8_t *plan_dev;
    uint32_t ntiles;
    uint32_t grid;
    uint32_t npes, all_total;
    size_t tiles_off, done_off, arrive_off, trace_off;
    uint32_t stage_bytes, nstages;
    bool trace_on;
};

// ---------------------------------------------------------------------------------------------------------
// device
// ---------------------------------------------------------------------------------------------------------
struct Epoch { unsigned e, all_total, npes; };    // e = launch index mod 2^32

__device__ __forceinline__ void wait_deps(const unsigned *done, const Epoch &ep, unsigned initiator, unsigned dep_pe,
                                          unsigned dep_all, unsigned pe_total) {
    if (dep_pe) while (ld_relaxed_u32(done + initiator) - ep.e * pe_total < dep_pe) __nanosleep(20);
    if (dep_all) while (ld_relaxed_u32(done + ep.npes) - ep.e * ep.all_total < dep_all) __nanosleep(20);
    if (dep_pe | dep_all) fence_acquire();
}

__device__ __forceinline__ void count_done(unsigned *done, unsigned npes, unsigned kind, unsigned initiator) {
    if (kind & TF_CNT_PE) red_release_add_u32(done + initiator, 1u);
    if (kind & TF_CNT_ALL) red_release_add_u32(done + npes, 1u);
}

// Completion accounting of one piece whose own writes are complete and visible to the calling thread.
__device__ __forceinline__ void account(const TileRec &r, unsigned *done, unsigned *arrive, const Epoch &ep) {
    if (!(r.kind & TF_ACCT)) return;
    if (r.nt > 1) {
        unsigned old;   // release: this piece's writes; acquire: the pieces that arrived earlier
        asm volatile("atom.acq_rel.gpu.global.add.u32 %0, [%1], 1;" : "=r"(old) : "l"(arrive + r.op) : "memory");
        if (old - ep.e * r.nt != r.nt - 1) return;                  // not the last piece of this launch to arrive
    }
    if (r.kind & TF_SIGNAL) signal_update(reinterpret_cast<unsigned long long *>(r.sig), r.value, (r.kind >> 8) & 0xff);
    count_done(done, ep.npes, r.kind, r.initiator);
}

__device__ __forceinline__ void amo_one(const AuxRec &o) {
    unsigned long long *word = reinterpret_cast<unsigned long long *>(o.word);
    const unsigned opc = o.kind & 0xffu;
    if (opc == SHMEMG_OP_ATOMIC_ADD) {
        asm volatile("red.relaxed.gpu.global.add.u64 [%0], %1;" ::"l"(word), "l"(o.value) : "memory");
    } else if (opc == SHMEMG_OP_ATOMIC_FETCH_ADD) {
        unsigned long long old = atomicAdd(word, (unsigned long long)o.value);
        *reinterpret_cast<volatile unsigned long long *>(o.fetch) = old;
    } else {
        unsigned long long old = atomicCAS(word, (unsigned long long)o.cond, (unsigned long long)o.value);
        *reinterpret_cast<volatile unsigned long long *>(o.fetch) = old;
    }
}

template <typename T> __device__ __forceinline__ T ld_rec(const T *p) {     // 64-byte immutable plan record
    static_assert(sizeof(T) == 64, "64-byte records");
    T r;
    const int4 *s = reinterpret_cast<const int4 *>(p);
    int4 *d = reinterpret_cast<int4 *>(&r);
    // L2 loads (every record is read once, by one thread); not the read-only path: the plan of a one-call batch is written
    // by the planning kernel while this kernel's CTAs are already resident (programmatic dependent launch)
    d[0] = ld_stream16(s); d[1] = ld_stream16(s + 1); d[2] = ld_stream16(s + 2); d[3] = ld_stream16(s + 3);
    return r;
}

// SHMEMG_TRACE=1 at batch creation: every CTA stamps %globaltimer at its role milestones into the plan's trace region
__device__ __forceinline__ unsigned long long gtime() {
    unsigned long long t;
    asm volatile("mov.u64 %0, %globaltimer;" : "=l"(t));
    return t;
}
// (builds with -DSHMEMG_EXPERIMENTS only: the shipped kernel carries no stamps)
#ifdef SHMEMG_EXPERIMENTS
#define TRACE(slot) do { if (trace) trace[blockIdx.x * TRACE_SLOTS + (slot)] = gtime(); } while (0)
#else
#define TRACE(slot) do { } while (0)
#endif

__global__ void __launch_bounds__(EXEC_THREADS, 1) k_batch_exec(const ExecArgs a) {
    extern __shared__ __align__(1024) uint8_t stage[];
    __shared__ __align__(16) TileRec ringA[EXEC_STAGES_MAX];
    __shared__ __align__(16) TileRec ringG[GEN_SLOTS];
    __shared__ uint64_t fullA[EXEC_STAGES_MAX], emptyA[EXEC_STAGES_MAX], fullG[GEN_SLOTS], emptyG[GEN_SLOTS], epochB;
    __shared__ unsigned s_epoch;

    const TileRec *tiles = a.tiles;
    unsigned *done = a.done, *arrive = a.arrive;
    unsigned ntiles = a.ntiles;
    unsigned STG = a.stage_bytes, NST = a.nstages;
    const int tid = threadIdx.x;
#ifdef SHMEMG_EXPERIMENTS
    unsigned long long *trace = blockIdx.x < TRACE_CTAS ? a.trace : nullptr;
#endif
    Epoch ep;
    ep.e = 0; ep.all_total = a.all_total; ep.npes = a.npes;

    if (tid == 0) {
        TRACE(0);
        for (int s = 0; s < EXEC_STAGES_MAX; ++s) { mbar_init(&fullA[s], 1); mbar_init(&emptyA[s], 1); }
        for (int g = 0; g < GEN_SLOTS; ++g) { mbar_init(&fullG[g], 1); mbar_init(&emptyG[g], 1); }
        mbar_init(&epochB, 1);
        mbar_init_fence();
    }
    // every executor releases ITS dependents at once (a following executor or planner launch sets itself up while this one runs)
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    if (a.hdr) {
        // One-call batch (shmemg_enqueue_batch): the planning kernel is the previous kernel of the stream and this one is
        // launched as its programmatic dependent, so everything above overlaps the planner; from here on its writes
        // (header, tile records, zeroed counters) are visible.  Coherent (L2) loads: nothing of the plan is in L1 yet.
#ifdef SHMEMG_PLAN_TRACE
        if (blockIdx.x == 0 && tid == 0) const_cast<PlanHeader *>(a.hdr)->pad3[8] = gtime();
#endif
        asm volatile("griddepcontrol.wait;" ::: "memory");
#ifdef SHMEMG_PLAN_TRACE
        if (blockIdx.x == 0 && tid == 0) const_cast<PlanHeader *>(a.hdr)->pad3[9] = gtime();
#endif
        const int4 h0 = ld_stream16(&a.hdr->ntiles);            // ntiles, nunits, npes, trace_on
        const int4 h1 = ld_stream16(&a.hdr->stage_bytes);       // stage_bytes, nstages, status, pad
        const unsigned at = *reinterpret_cast<const volatile unsigned *>(&a.hdr->all_total);
        ntiles = h1.z == 0 ? (unsigned)h0.x : 0u;               // a rejected plan executes nothing
        STG = (unsigned)h1.x; NST = (unsigned)h1.y;
        ep.all_total = at;
    }
    // Pre-planned batch: every launch is a programmatic dependent of whatever kernel precedes it in the stream.  Its tile
    // records are immutable, so the loader's first record is requested now; nothing mutable (ticket, counters, signal
    // words, payload) is touched before griddepcontrol.wait, which returns when the preceding grid has completed and its
    // writes are visible.  The executor releases ITS dependents at once: a following executor launch sets up its CTAs
    // (as SMs become free) while this one still runs, and blocks in the same wait.
    TileRec r0 = {};
    if (!a.hdr) {
        if (tid == 0 && blockIdx.x < ntiles) r0 = ld_rec(tiles + blockIdx.x);
        asm volatile("griddepcontrol.wait;" ::: "memory");
    }
    __syncthreads();

    if (tid == 0) {
        // ---- loader -------------------------------------------------------------------------------------------
        // The first ticket of CTA b is b (no atomic on the critical path, and the first wave is spread over all CTAs);
        // later tickets are claimed one ahead, while the current piece is processed.
        // Launch index: this launch's claims keep the counter inside [epoch*ntiles, (epoch+1)*ntiles) until the last
        // CTA's failing claim, and a CTA reads it before making its own.  The read is a cold miss (about 1 us): it is
        // issued first and consumed only after the first segment's loads are in flight; the consumers pick s_epoch up
        // through the epochB mbarrier before their first completion accounting.
        TRACE(1);
        const unsigned long long tk0 = a.hdr ? 0ull : ld_relaxed_u64(a.ticket);   // one-call plans start at launch index 0
        if (a.hdr && blockIdx.x < ntiles) r0 = ld_rec(tiles + blockIdx.x);
        unsigned ia = 0, ig = 0;                                     // ia = stage index, pa = its lap parity
        unsigned pa = 0, nissued = 0;
        auto issue = [&](const TileRec &r, unsigned off) {
            const unsigned s = ia;
            const unsigned n = r.nbytes - off < STG ? r.nbytes - off : STG;
            mbar_wait(&emptyA[s], pa ^ 1u);                              // passes at once on the ring's first lap
            TileRec q = r;
            q.dst = r.dst + off; q.nbytes = n;
            if (off + n == r.nbytes) q.kind |= TF_SEGEND;
            ringA[s] = q;
            mbar_arrive_expect_tx(&fullA[s], n);
            bulk_g2s(stage + (size_t)s * STG, reinterpret_cast<const void *>(r.src + off), n, &fullA[s]);
            if (++ia == NST) { ia = 0; pa ^= 1u; }
            ++nissued;
        };
        unsigned pre = 0;                                            // bytes of r0 already issued
        if ((r0.kind & (0xffu | TF_DEPS)) == T_TMA) {                // no dependencies: start streaming before the epoch is known
            for (; pre < r0.nbytes && nissued < NST; pre += STG) issue(r0, pre);
            TRACE(6);
        }
        ep.e = (unsigned)(tk0 / ntiles);
        s_epoch = ep.e;
        mbar_arrive(&epochB);
        const unsigned long long tbase = (unsigned long long)ep.e * ntiles;   // exact: epoch < 2^32 launches
        unsigned long long t0 = blockIdx.x;
        while (t0 < ntiles) {
            const unsigned long long t1 = atomicAdd(a.ticket, 1ull) - tbase + gridDim.x;
            const unsigned k = r0.kind & 0xffu;
            if (r0.kind & TF_DEPS) {
                wait_deps(done, ep, r0.initiator, r0.dep_pe, r0.dep_all, r0.pe_total);
                proxy_fence();                                       // acquire (generic proxy) before bulk reads
            }
            if (k == T_TMA) {                                        // one segment: stream its bulk tiles
                for (unsigned off = pre; off < r0.nbytes; off += STG) issue(r0, off);
                pre = 0;
            } else if (k == T_COPY || k == T_AMO || k == T_WAIT) {   // generic warps (a wait run is polled one wait per thread)
                const unsigned g = ig % GEN_SLOTS;
                mbar_wait(&emptyG[g], ((ig / GEN_SLOTS) & 1u) ^ 1u);
                ringG[g] = r0;
                mbar_arrive(&fullG[g]);
                ig++;
            } else {                                                 // T_NODATA: zero-byte put/get/put_signal
                account(r0, done, arrive, ep);
            }
            t0 = t1;
            if (t0 < ntiles) r0 = ld_rec(tiles + t0);
        }
        TRACE(2);
        {   // end markers for both consumers
            const unsigned s = ia;
            mbar_wait(&emptyA[s], pa ^ 1u);
            ringA[s].kind = T_END;
            mbar_arrive(&fullA[s]);
            const unsigned g = ig % GEN_SLOTS;
            mbar_wait(&emptyG[g], ((ig / GEN_SLOTS) & 1u) ^ 1u);
            ringG[g].kind = T_END;
            mbar_arrive(&fullG[g]);
        }
    } else if (tid == 32) {
        // ---- storer -------------------------------------------------------------------------------------------
        bool have_prev = false, pend_acct = false;     // previous tile's stage not yet freed / segment not yet accounted
        bool have_epoch = false;
        TileRec acct = {};
        unsigned prev_s = 0;
        auto epoch = [&]() { if (!have_epoch) { mbar_wait(&epochB, 0); ep.e = s_epoch; have_epoch = true; } };
        for (unsigned i = 0, s = 0, ph = 0;; ++i) {
            if (!mbar_test_wait(&fullA[s], ph)) {
                if (have_prev) {              // starved: nothing may stay unaccounted while this role blocks
                    if (pend_acct) { bulk_wait<0>(); proxy_fence(); epoch(); account(acct, done, arrive, ep); pend_acct = false; }
                    else bulk_wait_read<0>();
                    mbar_arrive(&emptyA[prev_s]);
                    have_prev = false;
                }
                mbar_wait(&fullA[s], ph);
            }
            const TileRec r = ringA[s];
            if ((r.kind & 0xffu) == T_END) break;
            if (i == 0) TRACE(7);
            bulk_s2g(reinterpret_cast<void *>(r.dst), stage + (size_t)s * STG, r.nbytes);
            bulk_commit();
            if (have_prev) {
                // every group but the one just committed: has completed (a segment ended) / has read its stage
                if (pend_acct) { bulk_wait<1>(); proxy_fence(); epoch(); account(acct, done, arrive, ep); pend_acct = false; }
                else bulk_wait_read<1>();
                mbar_arrive(&emptyA[prev_s]);
            }
            if ((r.kind & TF_SEGEND) && (r.kind & TF_ACCT)) { acct = r; pend_acct = true; }
            prev_s = s; have_prev = true;
            if (++s == NST) { s = 0; ph ^= 1u; }
        }
        TRACE(3);
        bulk_wait<0>();
        if (pend_acct) { proxy_fence(); epoch(); account(acct, done, arrive, ep); }
        TRACE(4);
#ifdef SHMEMG_PLAN_TRACE
        if (a.hdr && blockIdx.x == 0) const_cast<PlanHeader *>(a.hdr)->pad3[10] = gtime();
#endif
    } else if (tid >= GEN_FIRST) {
        // ---- generic warps: register-path copies and AMO runs ----------------------------------------------
        const int gt = tid - GEN_FIRST;
        for (unsigned j = 0;; ++j) {
            const unsigned g = j % GEN_SLOTS;
            mbar_wait(&fullG[g], (j / GEN_SLOTS) & 1u);
            const TileRec r = ringG[g];
            const unsigned k = r.kind & 0xffu;
            if (k == T_END) break;
            if (j == 0) { mbar_wait(&epochB, 0); ep.e = s_epoch; }
            if (k == T_COPY) {
                copy_coop<4>(reinterpret_cast<uint8_t *>(r.dst), reinterpret_cast<const uint8_t *>(r.src), r.nbytes, gt,
                             GEN_THREADS);
                if (r.kind & TF_ACCT) __threadfence();
            } else if (k == T_WAIT) {
                // a run of consecutive waits (any PEs): thread i polls wait i and accounts for it on its own
                if (gt < (int)r.nbytes) {
                    const AuxRec o = ld_rec(reinterpret_cast<const AuxRec *>(r.src) + gt);
                    const unsigned long long *sig = reinterpret_cast<const unsigned long long *>(o.word);
                    const int cmp = (int)((o.kind >> 8) & 0xff);
                    wait_deps(done, ep, o.initiator, o.dep_pe, o.dep_all, o.pe_total);
                    for (unsigned spin = 0; !cmp_u64(cmp, ld_relaxed_u64(sig), o.value); ++spin)
                        if (spin > 64) __nanosleep(32);
                    if (o.kind & (TF_CNT_PE | TF_CNT_ALL)) {     // some later op of this launch follows the wait
                        fence_acquire();
                        count_done(done, ep.npes, o.kind, o.initiator);
                    }                                            // else: the end of the kernel orders everything after it
                }
            } else if (gt < (int)r.nbytes) {
                const AuxRec o = ld_rec(reinterpret_cast<const AuxRec *>(r.src) + gt);
                wait_deps(done, ep, o.initiator, o.dep_pe, o.dep_all, o.pe_total);
                amo_one(o);
                count_done(done, ep.npes, o.kind, o.initiator);
            }
            named_bar_sync(1, GEN_THREADS);
            if (gt == 0) {
                if (k == T_COPY) account(r, done, arrive, ep);
                mbar_arrive(&emptyG[g]);
            }
        }
        if (gt == 0) TRACE(5);
    }
}

// ---- single copy on a stream ------------------------------------------------------------------------------------
// bulk-copy path (16-byte aligned): one issuing thread per CTA; optional last-arriver signal
__global__ void __launch_bounds__(32) k_copy_single_tma(uint8_t *dst, const uint8_t *src, size_t nbytes,
                                                        unsigned long long *sig, unsigned long long sig_value, int sig_op,
                                                        unsigned *counter) {
    extern __shared__ __align__(1024) uint8_t stage[];
    __shared__ uint64_t full[SHMEMG_TMA_STAGES];
    if (threadIdx.x != 0) return;
    tma_stream_init(full);
    const size_t nitems = (nbytes + SHMEMG_TMA_TILE - 1) / SHMEMG_TMA_TILE;
    tma_stream_copy(stage, full, blockIdx.x, gridDim.x, nitems, [&](size_t k, const uint8_t *&s, uint8_t *&d, unsigned &n) {
        const size_t off = k * SHMEMG_TMA_TILE;
        s = src + off; d = dst + off;
        n = (unsigned)(nbytes - off < SHMEMG_TMA_TILE ? nbytes - off : SHMEMG_TMA_TILE);
    });
    if (sig) {
        proxy_fence();
        __threadfence();
        if (atomicAdd(counter, 1u) == gridDim.x - 1) {
            __threadfence();
            *counter = 0;
            signal_update(sig, sig_value, sig_op);
        }
    }
}
// register path (any alignment): grid-stride over tiles, optional last-arriver signal
__global__ void __launch_bounds__(SHMEMG_THREADS, 4)
k_copy_single(uint8_t *dst, const uint8_t *src, size_t nbytes, unsigned tile_bytes, unsigned long long *sig,
              unsigned long long sig_value, int sig_op, unsigned *counter) {
    const size_t ntiles = (nbytes + tile_bytes - 1) / tile_bytes;
    for (size_t t = blockIdx.x; t < ntiles; t += gridDim.x) {
        const size_t off = t * tile_bytes;
        size_t n = nbytes - off;
        if (n > tile_bytes) n = tile_bytes;
        copy_coop<8>(dst + off, src + off, n, threadIdx.x, SHMEMG_THREADS);
    }
    if (sig) {
        __syncthreads();
        if (threadIdx.x == 0) {
            __threadfence();
            if (atomicAdd(counter, 1u) == gridDim.x - 1) {
                __threadfence();
                *counter = 0;
                signal_update(sig, sig_value, sig_op);
            }
        }
    }
}

__global__ void k_wait_until(const unsigned long long *sig, int cmp, unsigned long long value) {
    while (!cmp_u64(cmp, ld_relaxed_u64(sig), value)) __nanosleep(100);
    fence_acquire();
}

// ---------------------------------------------------------------------------------------------------------
// host: validation + planning
// ---------------------------------------------------------------------------------------------------------
int shmemg_validate_op(const shmemg_world *w, const shmemg_op_t &o) {
    switch (o.opcode) {
    case SHMEMG_OP_FENCE: case SHMEMG_OP_QUIET:
        if (o.ctx >= SHMEMG_CTX_MAX) return SHMEMG_ERR_ARG;
        return shmemg_pe_ok(w, o.initiator_pe) ? SHMEMG_OK : SHMEMG_ERR_PE;
    case SHMEMG_OP_BARRIER_ALL:
        return SHMEMG_OK;
    default: break;
    }
    if (o.opcode < SHMEMG_OP_PUT || o.opcode > SHMEMG_OP_BARRIER_ALL) return SHMEMG_ERR_ARG;
    if (o.ctx >= SHMEMG_CTX_MAX) return SHMEMG_ERR_ARG;
    if (!shmemg_pe_ok(w, o.initiator_pe)) return SHMEMG_ERR_PE;
    if (o.opcode == SHMEMG_OP_SIGNAL_WAIT_UNTIL) {
        if (o.cmp > SHMEMG_CMP_LE) return SHMEMG_ERR_ARG;
        if (!shmemg_in_range(w, o.loc_off, 8)) return SHMEMG_ERR_RANGE;
        return (o.loc_off & 7) ? SHMEMG_ERR_ALIGN : SHMEMG_OK;
    }
    if (!shmemg_pe_ok(w, o.target_pe)) return SHMEMG_ERR_PE;
    if (o.opcode <= SHMEMG_OP_PUT_SIGNAL) {
        if (!shmemg_in_range(w, o.rem_off, o.nbytes) || !shmemg_in_range(w, o.loc_off, o.nbytes)) return SHMEMG_ERR_RANGE;
        if (o.opcode == SHMEMG_OP_PUT_SIGNAL) {
            if (o.sig_op > SHMEMG_SIGNAL_ADD) return SHMEMG_ERR_ARG;
            if (!shmemg_in_range(w, o.sig_off, 8)) return SHMEMG_ERR_RANGE;
            if (o.sig_off & 7) return SHMEMG_ERR_ALIGN;
        }
        return SHMEMG_OK;
    }
    // AMOs
    if (!shmemg_in_range(w, o.rem_off, 8)) return SHMEMG_ERR_RANGE;
    if (o.rem_off & 7) return SHMEMG_ERR_ALIGN;
    if (o.opcode != SHMEMG_OP_ATOMIC_ADD) {
        if (!shmemg_in_range(w, o.loc_off, 8)) return SHMEMG_ERR_RANGE;
        if (o.loc_off & 7) return SHMEMG_ERR_ALIGN;
    }
    return SHMEMG_OK;
}

static bool is_marker(uint8_t opc) {
    return opc == SHMEMG_OP_FENCE || opc == SHMEMG_OP_QUIET || opc == SHMEMG_OP_BARRIER_ALL;
}
static bool is_amo(uint8_t opc) { return opc >= SHMEMG_OP_ATOMIC_ADD && opc <= SHMEMG_OP_ATOMIC_COMPARE_SWAP; }


// Cut one copy op into (kind, offset, bytes) pieces.  Source and destination congruent mod 16: unaligned head and
// tail go to the register path, the aligned body to bulk-copy tiles; otherwise register-path tiles throughout.
struct Piece { uint32_t kind; uint64_t off; uint32_t n; };
static void cut_copy(uint64_t dst, uint64_t src, uint64_t n, uint32_t seg_tiles, std::vector<Piece> &out) {
    out.clear();
    if (n == 0) { out.push_back({T_NODATA, 0, 0}); return; }
    const bool congruent = ((dst ^ src) & 15) == 0;
    const bool aligned = congruent && (dst & 15) == 0 && (n & 15) == 0;
    if (aligned || (congruent && n >= TMA_MIN_SPLIT)) {
        uint64_t head = (16 - (dst & 15)) & 15;
        if (head > n) head = n;
        const uint64_t body = (n - head) & ~15ull, tail = n - head - body;
        if (head) out.push_back({T_COPY, 0, (uint32_t)head});
        // balanced segments of at most seg_tiles bulk tiles
        const uint64_t tiles = (body + SHMEMG_TMA_TILE - 1) / SHMEMG_TMA_TILE;
        const uint64_t nseg = (tiles + seg_tiles - 1) / seg_tiles;
        // equal byte shares, cut at 1 KiB (the executor re-tiles a segment); one division per op: the device planner
        // (plan_dev.cu) applies the same rule
        const uint64_t share = ((body + nseg - 1) / nseg + 1023ull) & ~1023ull;
        for (uint64_t b0 = 0; b0 < body; b0 += share)
            out.push_back({T_TMA, head + b0, (uint32_t)(body - b0 < share ? body - b0 : share)});
        if (tail) out.push_back({T_COPY, head + body, (uint32_t)tail});
        return;
    }
    for (uint64_t o = 0; o < n; o += GEN_TILE) out.push_back({T_COPY, o, (uint32_t)(n - o < GEN_TILE ? n - o : GEN_TILE)});
}

// Segment length: a small batch is cut so that every SM gets about one segment (one completion fence per CTA);
// a large batch uses the maximum (dynamic tickets balance it).
static uint32_t pick_seg_tiles(const shmemg_world *w, const shmemg_op_t *ops, size_t nops) {
    uint64_t tiles = 0;
    for (size_t i = 0; i < nops; ++i)
        if (ops[i].opcode >= SHMEMG_OP_PUT && ops[i].opcode <= SHMEMG_OP_PUT_SIGNAL)
            tiles += (ops[i].nbytes + SHMEMG_TMA_TILE - 1) / SHMEMG_TMA_TILE;
    const uint64_t per_sm = (tiles + w->sm_count - 1) / w->sm_count;
#ifdef SHMEMG_EXPERIMENTS
    if (const char *e = getenv("SHMEMG_SEG_TILES")) {             // host planner only: plans then differ from the device planner's
        const int v = atoi(e);
        return v < 1 ? 1u : v > (int)SEG_TILES_MAX ? SEG_TILES_MAX : (uint32_t)v;
    }
#endif
    if (per_sm >= SEG_TILES_MAX) return SEG_TILES_MAX;
    return per_sm < 1 ? 1u : (uint32_t)per_sm;
}

// Per-op segment length.  Streaming batches: tickets are claimed in batch order, so whoever claims a 256 KiB segment last
// works alone for microseconds while the other SMs idle; the copy ops that start within the last `sm_count * 8` planner
// tiles (37 MB) of a streaming batch are therefore cut into 64 KiB segments (C3b 71.2 -> 68.6 us).
#define SEG_TILES_TAIL 2u
static void seg_tiles_per_op(const shmemg_world *w, const shmemg_op_t *ops, size_t nops, std::vector<uint32_t> &seg) {
    const uint32_t base = pick_seg_tiles(w, ops, nops);
    seg.assign(nops, base);
    if (base < SEG_TILES_MAX) return;
    uint64_t tiles = 0;
    const uint64_t tail = (uint64_t)w->sm_count * 8;      // measured on C3b: (8, 2) 68.6 us; (8, 1) 69.6; (16, 2) 69.1; (32, 2) 70.7; none 71.2
    const uint32_t tseg = SEG_TILES_TAIL;
    for (size_t i = nops; i-- > 0;) {
        if (ops[i].opcode < SHMEMG_OP_PUT || ops[i].opcode > SHMEMG_OP_PUT_SIGNAL) continue;
        if (tiles >= tail) break;
        seg[i] = tseg;
        tiles += (ops[i].nbytes + SHMEMG_TMA_TILE - 1) / SHMEMG_TMA_TILE;
    }
}

// ---- planning units: one per op (a marker, a copy op, an AMO, a wait) -------------------------------------------------
struct Unit { uint8_t opc; int pe; size_t first, count; };    // [first, first+count) in the caller's op array

// Ordering domains: FENCE / QUIET / SIGNAL_WAIT_UNTIL order the ops of ONE (PE, context) pair (a
// context is an independent ordering domain); domain index = ctx * npes + pe.  Unit.pe holds that index.
static int count_domains(const shmemg_world *w, const shmemg_op_t *ops, size_t nops) {
    int nctx = 1;
    for (size_t i = 0; i < nops; ++i)
        if (ops[i].opcode != SHMEMG_OP_BARRIER_ALL && ops[i].ctx + 1 > nctx) nctx = ops[i].ctx + 1;
    return nctx * w->npes;
}
static void build_units(const shmemg_world *w, const shmemg_op_t *ops, size_t nops, std::vector<Unit> &units) {
    units.clear();
    for (size_t i = 0; i < nops; ++i) {
        const shmemg_op_t &o = ops[i];
        units.push_back({o.opcode, o.opcode == SHMEMG_OP_BARRIER_ALL ? 0 : o.initiator_pe + (int)o.ctx * w->npes, i, 1});
    }
}

struct PlanSizes { size_t nunits, naux, ntiles, total; size_t tiles_off, aux_off, done_off, arrive_off, trace_off; };

static void copy_endpoints(const shmemg_world *w, const shmemg_op_t &o, uint64_t &dst, uint64_t &src) {
    const bool put = o.opcode != SHMEMG_OP_GET;
    dst = (uint64_t)shmemg_addr(w, put ? o.target_pe : o.initiator_pe, put ? o.rem_off : o.loc_off);
    src = (uint64_t)shmemg_addr(w, put ? o.initiator_pe : o.target_pe, put ? o.loc_off : o.rem_off);
}

static PlanSizes plan_sizes(const shmemg_world *w, const shmemg_op_t *ops, size_t nops, const std::vector<Unit> &units) {
    PlanSizes s{};
    size_t run = 0;
    uint32_t run_kind = 0;
    std::vector<Piece> pieces;
    std::vector<uint32_t> seg_tiles;
    seg_tiles_per_op(w, ops, nops, seg_tiles);
    for (const Unit &u : units) {
        if (is_marker(u.opc)) { run = 0; continue; }
        s.nunits++;
        if (is_amo(u.opc) || u.opc == SHMEMG_OP_SIGNAL_WAIT_UNTIL) {     // runs of AMOs / runs of waits: one tile each
            const uint32_t rk = is_amo(u.opc) ? T_AMO : T_WAIT;
            s.naux++;
            if (run == 0 || run == AMO_RUN_MAX || rk != run_kind || u.first % PLAN_CHUNK_OPS == 0) { s.ntiles++; run = 0; run_kind = rk; }
            run++;
            continue;
        }
        run = 0;
        uint64_t dst, src;
        copy_endpoints(w, ops[u.first], dst, src);
        cut_copy(dst, src, ops[u.first].nbytes, seg_tiles[u.first], pieces);
        s.ntiles += pieces.size();
    }
    auto up = [](size_t x) { return (x + 255) / 256 * 256; };
    s.tiles_off = sizeof(PlanHeader);
    s.aux_off = s.tiles_off + up(s.ntiles * sizeof(TileRec));
    s.done_off = s.aux_off + up(s.naux * sizeof(AuxRec));
    s.arrive_off = s.done_off + up(((size_t)count_domains(w, ops, nops) + 1) * 4);
    s.trace_off = s.arrive_off + up(s.nunits * 4);
    s.total = s.trace_off + TRACE_BYTES;
    return s;
}

extern "C" size_t shmemg_batch_plan_bytes(const shmemg_world_t *w, const shmemg_op_t *ops_host, size_t nops) {
    if (!w || (!ops_host && nops)) return 0;
    // an invalid descriptor is reported (with its index) by shmemg_batch_create, which never touches the plan then
    for (size_t i = 0; i < nops; ++i)
        if (shmemg_validate_op(w, ops_host[i])) return sizeof(PlanHeader);
    std::vector<Unit> units;
    build_units(w, ops_host, nops, units);
    return plan_sizes(w, ops_host, nops, units).total;
}

extern "C" int shmemg_batch_create(shmemg_world_t *w, const shmemg_op_t *ops, size_t nops, void *plan_dev,
                                   size_t plan_bytes, void *stream, shmemg_batch_t **out, size_t *bad_index) {
    if (!w || !out || !plan_dev || (!ops && nops)) return SHMEMG_ERR_ARG;
    *out = nullptr;
    if ((uintptr_t)plan_dev % 256) return SHMEMG_ERR_ALIGN;
    for (size_t i = 0; i < nops; ++i) {
        int rc = shmemg_validate_op(w, ops[i]);
        if (rc) {
            if (bad_index) *bad_index = i;
            return rc;
        }
    }
    std::vector<Unit> units;
    build_units(w, ops, nops, units);
    const PlanSizes ps = plan_sizes(w, ops, nops, units);
    if (plan_bytes < ps.total) return SHMEMG_ERR_NOMEM;
    if (ps.ntiles >= 0xffffffffull || ps.nunits >= 0xffffffffull) return SHMEMG_ERR_NOMEM;
    const size_t nu = units.size();

    // backward pass: which units does a LATER REAL unit depend on through a marker (or a wait)?
    std::vector<uint8_t> cnt(nu, 0);            // bit 0: count on done[initiator]; bit 1: count on done[npes]
    const int ndom = count_domains(w, ops, nops);
    std::vector<uint32_t> pe_total(ndom, 0);    // how far done[domain] advances per launch
    uint32_t all_total = 0;
    {
        std::vector<uint8_t> later_real(ndom, 0), later_nonwait(ndom, 0), need(ndom, 0);
        bool later_any = false, need_all = false;
        for (size_t i = nu; i-- > 0;) {
            const Unit &u = units[i];
            if (u.opc == SHMEMG_OP_FENCE || u.opc == SHMEMG_OP_QUIET) {
                if (later_real[u.pe]) need[u.pe] = 1;
                continue;
            }
            if (u.opc == SHMEMG_OP_BARRIER_ALL) { if (later_any) need_all = true; continue; }
            // a wait orders the domain's later ops after it: the wait and every earlier op of the domain are counted if
            // an op other than a wait follows (waits that only other waits follow order nothing: the end of the kernel does)
            if (u.opc == SHMEMG_OP_SIGNAL_WAIT_UNTIL && later_nonwait[u.pe]) need[u.pe] = 1;
            cnt[i] = (need[u.pe] ? 1 : 0) | (need_all ? 2 : 0);
            if (cnt[i] & 1) pe_total[u.pe]++;
            if (cnt[i] & 2) all_total++;
            later_real[u.pe] = 1;
            if (u.opc != SHMEMG_OP_SIGNAL_WAIT_UNTIL) later_nonwait[u.pe] = 1;
            later_any = true;
        }
    }

    std::vector<uint8_t> host(ps.total, 0);
    PlanHeader *hdr = reinterpret_cast<PlanHeader *>(host.data());
    TileRec *tiles = reinterpret_cast<TileRec *>(host.data() + ps.tiles_off);
    AuxRec *aux = reinterpret_cast<AuxRec *>(host.data() + ps.aux_off);
    hdr->ntiles = (uint32_t)ps.ntiles;
    hdr->nunits = (uint32_t)ps.nunits;
    hdr->npes = (uint32_t)ndom;
    hdr->all_total = all_total;
    hdr->tiles_off = ps.tiles_off; hdr->aux_off = ps.aux_off; hdr->done_off = ps.done_off; hdr->arrive_off = ps.arrive_off;
    hdr->trace_off = ps.trace_off;
#ifdef SHMEMG_EXPERIMENTS
    if (const char *e = getenv("SHMEMG_TRACE")) hdr->trace_on = (uint32_t)atoi(e);
#endif

    // forward pass: dependencies.  issued[p] = counted units of PE p so far; thresh[p] = what p's next unit must see.
    // (Only counted units advance done[], and every unit before a marker that a later unit depends on is counted.)
    // Consecutive waits of one PE (no other unit of that PE between them) share the threshold that was in force when the
    // run began, so they are polled concurrently; the threshold moves past the whole run at the PE's next unit
    // (wait_run[p]).  A wait must NOT get a weaker threshold than that: done[p] counts completions in any order, and
    // "done[p] >= issued-before-marker" means "everything before the marker is complete" only if nothing after the
    // marker can count before the marker's threshold is reached.
    std::vector<uint32_t> issued(ndom, 0), thresh(ndom, 0);
    std::vector<uint8_t> wait_run(ndom, 0);
    uint32_t all_issued = 0, all_thresh = 0, run_kind = 0;
    size_t k = 0, nt = 0, na = 0, run = 0;
    std::vector<Piece> pieces;
    std::vector<uint32_t> seg_tiles;
    seg_tiles_per_op(w, ops, nops, seg_tiles);
    auto aux_dev = [&](size_t idx) { return (uint64_t)((uint8_t *)plan_dev + ps.aux_off + idx * sizeof(AuxRec)); };
    for (size_t ui = 0; ui < nu; ++ui) {
        const Unit &u = units[ui];
        const shmemg_op_t &o = ops[u.first];
        if (u.opc == SHMEMG_OP_FENCE || u.opc == SHMEMG_OP_QUIET) { thresh[u.pe] = issued[u.pe]; wait_run[u.pe] = 0; run = 0; continue; }
        if (u.opc == SHMEMG_OP_BARRIER_ALL) { all_thresh = all_issued; run = 0; continue; }
        const int ini = u.pe;
        const uint32_t flags = ((cnt[ui] & 1) ? TF_CNT_PE : 0) | ((cnt[ui] & 2) ? TF_CNT_ALL : 0);
        if (wait_run[ini] && u.opc != SHMEMG_OP_SIGNAL_WAIT_UNTIL) { thresh[ini] = issued[ini]; wait_run[ini] = 0; }
        const uint32_t dep_pe = thresh[ini], dep_all = all_thresh;
        if (is_amo(u.opc)) {
            AuxRec &d = aux[na];
            d.word = (uint64_t)shmemg_addr(w, o.target_pe, o.rem_off);
            d.fetch = u.opc == SHMEMG_OP_ATOMIC_ADD ? 0 : (uint64_t)shmemg_addr(w, o.initiator_pe, o.loc_off);   // the PE, not the domain
            d.value = o.value; d.cond = o.cond;
            d.kind = u.opc | flags;
            d.initiator = (uint32_t)ini; d.dep_pe = dep_pe; d.dep_all = dep_all; d.pe_total = pe_total[ini];
            if (run == 0 || run == AMO_RUN_MAX || run_kind != T_AMO || u.first % PLAN_CHUNK_OPS == 0) {
                TileRec &t = tiles[nt++];
                t.kind = T_AMO; t.nbytes = 0; t.nt = 1; t.op = (uint32_t)k;
                t.src = aux_dev(na);
                run = 0; run_kind = T_AMO;
            }
            tiles[nt - 1].nbytes++;
            run++; na++;
        } else if (u.opc == SHMEMG_OP_SIGNAL_WAIT_UNTIL) {
            AuxRec &d = aux[na];
            d.word = (uint64_t)shmemg_addr(w, o.initiator_pe, o.loc_off);
            d.value = o.value;
            d.kind = SHMEMG_OP_SIGNAL_WAIT_UNTIL | ((uint32_t)o.cmp << 8) | flags;
            d.initiator = (uint32_t)ini; d.dep_pe = dep_pe; d.dep_all = dep_all; d.pe_total = pe_total[ini];
            if (run == 0 || run == WAIT_RUN_MAX || run_kind != T_WAIT || u.first % PLAN_CHUNK_OPS == 0) {
                TileRec &t = tiles[nt++];
                t.kind = T_WAIT; t.nbytes = 0; t.nt = 1; t.op = (uint32_t)k;
                t.src = aux_dev(na);
                run = 0; run_kind = T_WAIT;
            }
            tiles[nt - 1].nbytes++;
            run++; na++;
        } else {
            run = 0;
            uint64_t dst, src;
            copy_endpoints(w, o, dst, src);
            cut_copy(dst, src, o.nbytes, seg_tiles[u.first], pieces);
            uint32_t f = flags | ((dep_pe | dep_all) ? TF_DEPS : 0);
            uint64_t sig = 0;
            if (u.opc == SHMEMG_OP_PUT_SIGNAL) {
                f |= TF_SIGNAL | ((uint32_t)o.sig_op << 8);
                sig = (uint64_t)shmemg_addr(w, o.target_pe, o.sig_off);
            }
            for (size_t p = 0; p < pieces.size(); ++p) {
                TileRec &t = tiles[nt++];
                t.dst = dst + pieces[p].off; t.src = src + pieces[p].off; t.nbytes = pieces[p].n;
                t.kind = pieces[p].kind | f;
                t.sig = sig; t.value = o.value;
                t.op = (uint32_t)k; t.nt = (uint32_t)pieces.size(); t.initiator = (uint32_t)ini;
                t.dep_pe = dep_pe; t.dep_all = dep_all; t.pe_total = pe_total[ini];
            }
        }
        if (cnt[ui] & 1) issued[ini]++;
        if (cnt[ui] & 2) all_issued++;
        if (u.opc == SHMEMG_OP_SIGNAL_WAIT_UNTIL) wait_run[ini] = 1;           // later ops of this PE follow the run of waits
        k++;
    }

    cudaStream_t st = (cudaStream_t)stream;
    SHMEMG_CUDA(w, cudaMemcpyAsync(plan_dev, host.data(), ps.total, cudaMemcpyHostToDevice, st));
    SHMEMG_CUDA(w, cudaStreamSynchronize(st));

    shmemg_batch *b = new shmemg_batch();
    b->w = w;
    b->plan_dev = (uint8_t *)plan_dev;
    b->ntiles = (uint32_t)ps.ntiles;
    const uint64_t maxgrid = (uint64_t)w->sm_count;
    b->grid = (uint32_t)(ps.ntiles < maxgrid ? (ps.ntiles ? ps.ntiles : 1) : maxgrid);
    b->npes = (uint32_t)ndom; b->all_total = all_total;          // index of the all-domains counter in done[]
    b->tiles_off = ps.tiles_off; b->done_off = ps.done_off; b->arrive_off = ps.arrive_off; b->trace_off = ps.trace_off;
    b->trace_on = hdr->trace_on != 0;
    {
        uint64_t bulk = 0;
        for (size_t i = 0; i < nops; ++i)
            if (ops[i].opcode >= SHMEMG_OP_PUT && ops[i].opcode <= SHMEMG_OP_PUT_SIGNAL) bulk += ops[i].nbytes;
        const bool small = bulk <= (uint64_t)EXEC_SMALL_PER_SM * (uint64_t)w->sm_count;
        b->stage_bytes = small ? 16384u : 32768u;
        b->nstages = small ? 12u : 7u;
#ifdef SHMEMG_EXPERIMENTS
        if (const char *e = getenv("SHMEMG_EXEC_RING")) {            // "<stage_bytes>x<nstages>"
            unsigned sb = 0, ns = 0;
            if (sscanf(e, "%ux%u", &sb, &ns) == 2 && sb >= 1024 && sb % 16 == 0 && ns >= 2 && ns <= EXEC_STAGES_MAX &&
                (uint64_t)sb * ns <= EXEC_SMEM_MAX) { b->stage_bytes = sb; b->nstages = ns; }
        }
#endif
    }
    *out = b;
    return SHMEMG_OK;
}

extern "C" int shmemg_batch_destroy(shmemg_batch_t *b) {
    if (!b) return SHMEMG_ERR_ARG;
    delete b;
    return SHMEMG_OK;
}
extern "C" int shmemg_batch_launches(const shmemg_batch_t *b) { return b ? (b->ntiles ? 1 : 0) : SHMEMG_ERR_ARG; }

int shmemg_exec_smem_attr(shmemg_world *w) {
    if (w->smem_attr_set) return SHMEMG_OK;
    SHMEMG_CUDA(w, cudaFuncSetAttribute(k_batch_exec, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)EXEC_SMEM_MAX));
    SHMEMG_CUDA(w, cudaFuncSetAttribute(k_copy_single_tma, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SHMEMG_TMA_SMEM));
    w->smem_attr_set = true;
    return SHMEMG_OK;
}

// Launch the executor, always as a programmatic dependent of the kernel before it (programmatic stream serialization): when
// that kernel releases its dependents early (the device planner and every executor do, at entry), the executor's CTAs are set
// up while it still runs and block in griddepcontrol.wait until it has finished and its writes are visible; behind an ordinary
// kernel nothing changes.  after_planner only documents the call site (one-call form).
int shmemg_exec_launch(shmemg_world *w, const ExecArgs &a, unsigned grid, size_t smem, cudaStream_t st, bool after_planner) {
    int rc = shmemg_exec_smem_attr(w);
    if (rc) return rc;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(grid); cfg.blockDim = dim3(EXEC_THREADS); cfg.dynamicSmemBytes = smem; cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    (void)after_planner;
    cfg.attrs = at; cfg.numAttrs = w->dependent_launch ? 1 : 0;        // shmemg_set_dependent_launch
    SHMEMG_CUDA(w, cudaLaunchKernelEx(&cfg, k_batch_exec, a));
    return SHMEMG_OK;
}

extern "C" int shmemg_batch_enqueue_on_stream(shmemg_world_t *w, shmemg_batch_t *b, void *stream) {
    if (!w || !b || b->w != w) return SHMEMG_ERR_ARG;
    if (b->ntiles == 0) return SHMEMG_OK;
    ExecArgs a;
    a.tiles = reinterpret_cast<const TileRec *>(b->plan_dev + b->tiles_off);
    a.ticket = &reinterpret_cast<PlanHeader *>(b->plan_dev)->ticket;
    a.done = reinterpret_cast<unsigned *>(b->plan_dev + b->done_off);
    a.arrive = reinterpret_cast<unsigned *>(b->plan_dev + b->arrive_off);
    a.trace = b->trace_on ? reinterpret_cast<unsigned long long *>(b->plan_dev + b->trace_off) : nullptr;
    a.ntiles = b->ntiles; a.npes = b->npes; a.all_total = b->all_total;
    a.stage_bytes = b->stage_bytes; a.nstages = b->nstages;
    a.hdr = nullptr;
    return shmemg_exec_launch(w, a, b->grid, (size_t)b->stage_bytes * b->nstages, (cudaStream_t)stream, false);
}

// ---------------------------------------------------------------------------------------------------------
// single operations on a stream
// ---------------------------------------------------------------------------------------------------------
static int launch_copy(shmemg_world *w, uint8_t *dst, const uint8_t *src, size_t nbytes, unsigned long long *sig,
                       uint64_t sig_value, int sig_op, cudaStream_t st) {
    if (nbytes == 0 && !sig) return SHMEMG_OK;
    unsigned *counter = sig ? &w->ctl->sig_counter[(w->sig_seq++) % SHMEMG_SIG_SLOTS] : nullptr;
    if (nbytes && (((uintptr_t)dst | (uintptr_t)src | nbytes) & 15) == 0 && !w->tile_bytes_override) {
        int rc = shmemg_exec_smem_attr(w);
        if (rc) return rc;
        const uint64_t ntiles = (nbytes + SHMEMG_TMA_TILE - 1) / SHMEMG_TMA_TILE;
        const uint32_t grid = (uint32_t)(ntiles < (uint64_t)w->sm_count ? ntiles : (uint64_t)w->sm_count);
        k_copy_single_tma<<<grid, 32, SHMEMG_TMA_SMEM, st>>>(dst, src, nbytes, sig, sig_value, sig_op, counter);
        SHMEMG_CUDA(w, cudaGetLastError());
        return SHMEMG_OK;
    }
    const uint64_t maxgrid = (uint64_t)w->sm_count * w->ctas_per_sm;
    uint32_t tb = 8192;
    while (tb < 65536 && nbytes / tb > maxgrid * 8) tb <<= 1;
    if (w->tile_bytes_override) tb = (uint32_t)w->tile_bytes_override;
    uint64_t ntiles = (nbytes + tb - 1) / tb;
    uint32_t grid = (uint32_t)(ntiles < maxgrid ? (ntiles ? ntiles : 1) : maxgrid);
    k_copy_single<<<grid, SHMEMG_THREADS, 0, st>>>(dst, src, nbytes, tb, sig, sig_value, sig_op, counter);
    SHMEMG_CUDA(w, cudaGetLastError());
    return SHMEMG_OK;
}

extern "C" int shmemg_put_on_stream(shmemg_world_t *w, uint64_t dest_off, uint64_t source_off, size_t nbytes, int pe,
                                    int target_pe, void *stream) {
    if (!w) return SHMEMG_ERR_ARG;
    if (!shmemg_pe_ok(w, pe) || !shmemg_pe_ok(w, target_pe)) return SHMEMG_ERR_PE;
    if (!shmemg_in_range(w, dest_off, nbytes) || !shmemg_in_range(w, source_off, nbytes)) return SHMEMG_ERR_RANGE;
    return launch_copy(w, shmemg_addr(w, target_pe, dest_off), shmemg_addr(w, pe, source_off), nbytes, nullptr, 0, 0,
                       (cudaStream_t)stream);
}
extern "C" int shmemg_get_on_stream(shmemg_world_t *w, uint64_t dest_off, uint64_t source_off, size_t nbytes, int pe,
                                    int target_pe, void *stream) {
    if (!w) return SHMEMG_ERR_ARG;
    if (!shmemg_pe_ok(w, pe) || !shmemg_pe_ok(w, target_pe)) return SHMEMG_ERR_PE;
    if (!shmemg_in_range(w, dest_off, nbytes) || !shmemg_in_range(w, source_off, nbytes)) return SHMEMG_ERR_RANGE;
    return launch_copy(w, shmemg_addr(w, pe, dest_off), shmemg_addr(w, target_pe, source_off), nbytes, nullptr, 0, 0,
                       (cudaStream_t)stream);
}
extern "C" int shmemg_put_signal_on_stream(shmemg_world_t *w, uint64_t dest_off, uint64_t source_off, size_t nbytes,
                                           uint64_t sig_off, uint64_t signal, int sig_op, int pe, int target_pe,
                                           void *stream) {
    if (!w || sig_op < SHMEMG_SIGNAL_SET || sig_op > SHMEMG_SIGNAL_ADD) return SHMEMG_ERR_ARG;
    if (!shmemg_pe_ok(w, pe) || !shmemg_pe_ok(w, target_pe)) return SHMEMG_ERR_PE;
    if (!shmemg_in_range(w, dest_off, nbytes) || !shmemg_in_range(w, source_off, nbytes) ||
        !shmemg_in_range(w, sig_off, 8))
        return SHMEMG_ERR_RANGE;
    if (sig_off & 7) return SHMEMG_ERR_ALIGN;
    return launch_copy(w, shmemg_addr(w, target_pe, dest_off), shmemg_addr(w, pe, source_off), nbytes,
                       (unsigned long long *)shmemg_addr(w, target_pe, sig_off), signal, sig_op, (cudaStream_t)stream);
}
extern "C" int shmemg_signal_wait_until_on_stream(shmemg_world_t *w, uint64_t sig_off, int cmp, uint64_t value, int pe,
                                                  void *stream) {
    if (!w || cmp < SHMEMG_CMP_EQ || cmp > SHMEMG_CMP_LE) return SHMEMG_ERR_ARG;
    if (!shmemg_pe_ok(w, pe)) return SHMEMG_ERR_PE;
    if (!shmemg_in_range(w, sig_off, 8)) return SHMEMG_ERR_RANGE;
    if (sig_off & 7) return SHMEMG_ERR_ALIGN;
    k_wait_until<<<1, 1, 0, (cudaStream_t)stream>>>((const unsigned long long *)shmemg_addr(w, pe, sig_off), cmp, value);
    SHMEMG_CUDA(w, cudaGetLastError());
    return SHMEMG_OK;
}
extern "C" int shmemg_fence_on_stream(shmemg_world_t *w, int pe, void *stream) {
    (void)stream;
    if (!w) return SHMEMG_ERR_ARG;
    return shmemg_pe_ok(w, pe) ? SHMEMG_OK : SHMEMG_ERR_PE;
}
extern "C" int shmemg_quiet_on_stream(shmemg_world_t *w, int pe, void *stream) {
    return shmemg_fence_on_stream(w, pe, stream);
}
extern "C" int shmemg_quiet(shmemg_world_t *w, int pe, void *stream) {
    int rc = shmemg_fence_on_stream(w, pe, stream);
    if (rc) return rc;
    SHMEMG_CUDA(w, cudaStreamSynchronize((cudaStream_t)stream));
    return SHMEMG_OK;
}

// non-blocking forms on a stream: same kernels, weaker contract (see shmemg.h)
extern "C" int shmemg_put_nbi_on_stream(shmemg_world_t *w, uint64_t dest_off, uint64_t source_off, size_t nbytes, int pe,
                                        int target_pe, void *stream) {
    return shmemg_put_on_stream(w, dest_off, source_off, nbytes, pe, target_pe, stream);
}
extern "C" int shmemg_get_nbi_on_stream(shmemg_world_t *w, uint64_t dest_off, uint64_t source_off, size_t nbytes, int pe,
                                        int target_pe, void *stream) {
    return shmemg_get_on_stream(w, dest_off, source_off, nbytes, pe, target_pe, stream);
}
extern "C" int shmemg_put_signal_nbi_on_stream(shmemg_world_t *w, uint64_t dest_off, uint64_t source_off, size_t nbytes,
                                               uint64_t sig_off, uint64_t signal, int sig_op, int pe, int target_pe, void *stream) {
    return shmemg_put_signal_on_stream(w, dest_off, source_off, nbytes, sig_off, signal, sig_op, pe, target_pe, stream);
}
