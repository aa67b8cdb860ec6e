// plan_dev.cu -- the DEVICE PLANNER: shmemg_enqueue_batch, the one-call, host-initiated enqueue of a DEVICE-RESIDENT
// descriptor array on a stream ("internal GPU kernels to accelerate a host-issued
// or stream-triggered operation", L396).  No host pass over the descriptors, no synchronisation: the descriptors may have
// been produced by an earlier kernel of the stream (the graph workload's natural case).
//
//   k_plan_batch (1 CTA, or a cluster of 16 CTAs for more than 1024 ops; up to 512 threads each)  validates the descriptors, resolves PE -> address translation, cuts the copies into
//       tiles and writes EXACTLY the plan the host planner of batch.cu writes (same tile / AMO / wait records, same
//       dependency thresholds), so the same executor kernel runs both forms.  What the host does with two sequential passes
//       is done here with block-wide scans:
//         * which ops are counted (a later op of the (PE, context) domain depends on them through a FENCE / QUIET / wait, or
//           any later op through a BARRIER_ALL) follows from four maxima per domain -- last op, last op that is not a wait,
//           last marker a later op follows -- found with shared-memory atomicMax, no scan;
//         * tile-record / AMO-record / unit indices, the segment-length rule of streaming batches and the BARRIER_ALL
//           thresholds are prefix sums / prefix maxima over the op array (one op per thread, 512 ops per CTA, block totals
//           exchanged through distributed shared memory, a carry between super-chunks);
//         * the per-domain thresholds (counted ops of the domain before its latest FENCE / QUIET / end of a run of waits) are a
//           keyed prefix count: one warp walks the ops 32 at a time, ranks them inside their domain with match.any and
//           carries issued / threshold / in-a-run-of-waits per domain in shared memory.  It is skipped when no op is
//           counted and nothing depends on a marker (halo rounds, alltoall-style put batches).
//   k_batch_exec (batch.cu) is launched behind it as a programmatic dependent: its CTAs are set up while the planner runs and
//       read ntiles / ring geometry from the plan header once the planner has finished.
#include "batch_plan.cuh"

#ifndef PLAN_THREADS
#define PLAN_THREADS 512          // threads per planner CTA = ops per CTA and super-chunk: 128 registers per thread, no spills
#endif
#define PLAN_DOM_MAX 4096            // SHMEMG_CTX_MAX * npes the planner's shared-memory tables hold (npes <= 512)
#define FULLM 0xffffffffu

struct PlanArgs {
    const shmemg_op_t *ops;
    unsigned long long nops;
    uint8_t *base;                 // world
    unsigned long long stride, heap_bytes;
    int npes, sm_count;
    PlanHeader *hdr;               // workspace
    TileRec *tiles;
    AuxRec *aux;
    unsigned *done, *arrive;
    unsigned cap_tiles, ndom;
    unsigned long long tiles_off, aux_off, done_off, arrive_off;   // of the records inside the workspace (recorded in the header)
};

__device__ __forceinline__ bool d_in_range(unsigned long long off, unsigned long long n, unsigned long long heap) {
    return off <= heap && n <= heap - off;
}
__device__ __forceinline__ bool d_marker(unsigned opc) {
    return opc == SHMEMG_OP_FENCE || opc == SHMEMG_OP_QUIET || opc == SHMEMG_OP_BARRIER_ALL;
}
__device__ __forceinline__ bool d_amo(unsigned opc) { return opc >= SHMEMG_OP_ATOMIC_ADD && opc <= SHMEMG_OP_ATOMIC_COMPARE_SWAP; }
__device__ __forceinline__ bool d_copy(unsigned opc) { return opc >= SHMEMG_OP_PUT && opc <= SHMEMG_OP_PUT_SIGNAL; }
__device__ __forceinline__ unsigned d_class(unsigned opc) { return d_amo(opc) ? 1u : opc == SHMEMG_OP_SIGNAL_WAIT_UNTIL ? 2u : 0u; }

__device__ __forceinline__ shmemg_op_t d_ld_op(const shmemg_op_t *p) {
    shmemg_op_t r;
    const int4 *s = reinterpret_cast<const int4 *>(p);
    int4 *d = reinterpret_cast<int4 *>(&r);
    d[0] = ld_stream16(s); d[1] = ld_stream16(s + 1); d[2] = ld_stream16(s + 2); d[3] = ld_stream16(s + 3);
    return r;
}
// opcode / ctx / initiator only (first 16 bytes of the descriptor)
__device__ __forceinline__ void d_ld_head(const shmemg_op_t *p, unsigned &opc, unsigned &ctx, int &ini) {
    const int4 h = ld_stream16(p);
    opc = (unsigned)h.x & 0xffu; ctx = ((unsigned)h.x >> 24) & 0xffu; ini = h.y;
}

// the same checks as shmemg_validate_op (batch.cu), on the device
__device__ int d_validate(const PlanArgs &a, const shmemg_op_t &o) {
    const bool pe_ok = o.initiator_pe >= 0 && o.initiator_pe < a.npes;
    if (o.opcode == SHMEMG_OP_FENCE || o.opcode == SHMEMG_OP_QUIET) {
        if (o.ctx >= SHMEMG_CTX_MAX) return SHMEMG_ERR_ARG;
        return pe_ok ? SHMEMG_OK : SHMEMG_ERR_PE;
    }
    if (o.opcode == SHMEMG_OP_BARRIER_ALL) return SHMEMG_OK;
    if (o.opcode < SHMEMG_OP_PUT || o.opcode > SHMEMG_OP_BARRIER_ALL) return SHMEMG_ERR_ARG;
    if (o.ctx >= SHMEMG_CTX_MAX) return SHMEMG_ERR_ARG;
    if (!pe_ok) return SHMEMG_ERR_PE;
    if (o.opcode == SHMEMG_OP_SIGNAL_WAIT_UNTIL) {
        if (o.cmp > SHMEMG_CMP_LE) return SHMEMG_ERR_ARG;
        if (!d_in_range(o.loc_off, 8, a.heap_bytes)) return SHMEMG_ERR_RANGE;
        return (o.loc_off & 7) ? SHMEMG_ERR_ALIGN : SHMEMG_OK;
    }
    if (o.target_pe < 0 || o.target_pe >= a.npes) return SHMEMG_ERR_PE;
    if (o.opcode <= SHMEMG_OP_PUT_SIGNAL) {
        if (!d_in_range(o.rem_off, o.nbytes, a.heap_bytes) || !d_in_range(o.loc_off, o.nbytes, a.heap_bytes)) return SHMEMG_ERR_RANGE;
        if (o.opcode == SHMEMG_OP_PUT_SIGNAL) {
            if (o.sig_op > SHMEMG_SIGNAL_ADD) return SHMEMG_ERR_ARG;
            if (!d_in_range(o.sig_off, 8, a.heap_bytes)) return SHMEMG_ERR_RANGE;
            if (o.sig_off & 7) return SHMEMG_ERR_ALIGN;
        }
        return SHMEMG_OK;
    }
    if (!d_in_range(o.rem_off, 8, a.heap_bytes)) return SHMEMG_ERR_RANGE;
    if (o.rem_off & 7) return SHMEMG_ERR_ALIGN;
    if (o.opcode != SHMEMG_OP_ATOMIC_ADD) {
        if (!d_in_range(o.loc_off, 8, a.heap_bytes)) return SHMEMG_ERR_RANGE;
        if (o.loc_off & 7) return SHMEMG_ERR_ALIGN;
    }
    return SHMEMG_OK;
}

__device__ __forceinline__ void d_endpoints(const PlanArgs &a, const shmemg_op_t &o, unsigned long long &dst, unsigned long long &src) {
    const bool put = o.opcode != SHMEMG_OP_GET;
    const unsigned long long rem = (unsigned long long)(a.base + (size_t)o.target_pe * a.stride + o.rem_off);
    const unsigned long long loc = (unsigned long long)(a.base + (size_t)o.initiator_pe * a.stride + o.loc_off);
    dst = put ? rem : loc;
    src = put ? loc : rem;
}

// The cut of one copy op into pieces: the same rule as cut_copy (batch.cu), computed ONCE per op (the piece count feeds the
// scan, the pieces are emitted behind it).  Divisions run in 32 bits when the op is shorter than 4 GiB (a 64-bit division is
// about a hundred instructions, and the planner of a small batch is bound by instruction issue).
struct Cut {
    unsigned long long head, body, share;   // bulk mode: unaligned head, 16-byte body cut into `share`-byte pieces, tail
    unsigned tail, np, bulk;                // np = number of pieces; bulk = 0: register-path tiles of GEN_TILE bytes throughout
};
__device__ __forceinline__ Cut d_cut(unsigned long long dst, unsigned long long src, unsigned long long n, unsigned seg_tiles) {
    Cut c = {0, 0, 0, 0, 1, 0};
    if (n == 0) return c;                                            // one T_NODATA piece
    const bool congruent = ((dst ^ src) & 15) == 0;
    const bool aligned = congruent && (dst & 15) == 0 && (n & 15) == 0;
    if (aligned || (congruent && n >= TMA_MIN_SPLIT)) {
        unsigned long long head = (16 - (dst & 15)) & 15;
        if (head > n) head = n;
        const unsigned long long body = (n - head) & ~15ull;
        c.head = head; c.body = body; c.tail = (unsigned)(n - head - body); c.bulk = 1;
        const unsigned long long tiles = (body + SHMEMG_TMA_TILE - 1) / SHMEMG_TMA_TILE;
        unsigned nbody;
        if (body == 0) {
            nbody = 0;
        } else if ((body >> 32) == 0) {
            const unsigned t32 = (unsigned)tiles, b32 = (unsigned)body;
            const unsigned nseg = (t32 + seg_tiles - 1) / seg_tiles;                 // >= 1
            const unsigned q = b32 / nseg;
            const unsigned long long ceilq = (unsigned long long)q + (q * nseg != b32 ? 1u : 0u);
            c.share = (ceilq + 1023ull) & ~1023ull;                                  // equal shares, cut at 1 KiB
            if (c.share >> 32) nbody = 1u;
            else { const unsigned s32 = (unsigned)c.share, q2 = b32 / s32; nbody = q2 + (q2 * s32 != b32 ? 1u : 0u); }
        } else {
            const unsigned long long nseg = (tiles + seg_tiles - 1) / seg_tiles;
            c.share = ((body + nseg - 1) / nseg + 1023ull) & ~1023ull;
            nbody = (unsigned)((body + c.share - 1) / c.share);
        }
        c.np = (head ? 1u : 0u) + nbody + (c.tail ? 1u : 0u);
        return c;
    }
    c.np = (unsigned)((n + GEN_TILE - 1) / GEN_TILE);
    return c;
}
// emit(piece index, kind, offset, bytes) for every piece of the cut: ONE call site in a rolled loop (the record-writing code is
// the bulk of the planner's instructions, and the planner pays for every instruction line it fetches)
template <typename F>
__device__ __forceinline__ void d_emit_cut(const Cut &c, unsigned long long n, F emit) {
    const unsigned hp = c.head ? 1u : 0u, last = c.np - 1u;
#pragma unroll 1
    for (unsigned p = 0; p < c.np; ++p) {
        unsigned kind, len;
        unsigned long long off;
        if (n == 0) { kind = T_NODATA; off = 0; len = 0; }
        else if (!c.bulk) { kind = T_COPY; off = (unsigned long long)p * GEN_TILE; len = (unsigned)(n - off < GEN_TILE ? n - off : GEN_TILE); }
        else if (p < hp) { kind = T_COPY; off = 0; len = (unsigned)c.head; }
        else if (c.tail && p == last) { kind = T_COPY; off = c.head + c.body; len = c.tail; }
        else { const unsigned long long b0 = (unsigned long long)(p - hp) * c.share; kind = T_TMA; off = c.head + b0; len = (unsigned)(c.body - b0 < c.share ? c.body - b0 : c.share); }
        emit(p, kind, off, len);
    }
}

template <typename T> __device__ __forceinline__ void d_st_rec(T *p, const T &r) {       // 64-byte record, four 16-byte stores
    static_assert(sizeof(T) == 64, "64-byte records");
    const int4 *s = reinterpret_cast<const int4 *>(&r);
    int4 *d = reinterpret_cast<int4 *>(p);
    d[0] = s[0]; d[1] = s[1]; d[2] = s[2]; d[3] = s[3];
}

// ---- block-wide inclusive scan of (a, b, c: sums; m: maximum), up to 1024 threads ------------------------------------------------
struct S4 { unsigned a, b, c, m; };
__device__ __forceinline__ S4 s4_comb(const S4 &x, const S4 &y) { return {x.a + y.a, x.b + y.b, x.c + y.c, x.m > y.m ? x.m : y.m}; }
__device__ __forceinline__ S4 s4_shfl_up(const S4 &v, int o) {
    return {__shfl_up_sync(FULLM, v.a, o), __shfl_up_sync(FULLM, v.b, o), __shfl_up_sync(FULLM, v.c, o), __shfl_up_sync(FULLM, v.m, o)};
}
// returns the inclusive scan of v over the block; `total` = the block's combined value.  ws: 32 entries of shared memory.
__device__ __forceinline__ S4 block_scan(S4 v, S4 *ws, S4 &total) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarps = blockDim.x >> 5;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const S4 t = s4_shfl_up(v, o);
        if (lane >= o) v = s4_comb(t, v);
    }
    if (lane == 31) ws[warp] = v;
    __syncthreads();
    if (warp == 0) {
        S4 w = lane < nwarps ? ws[lane] : S4{0, 0, 0, 0};
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const S4 t = s4_shfl_up(w, o);
            if (lane >= o) w = s4_comb(t, w);
        }
        ws[lane] = w;
    }
    __syncthreads();
    if (warp > 0) v = s4_comb(ws[warp - 1], v);
    total = ws[31];                                   // lanes beyond the last warp carry the block total forward
    __syncthreads();
    return v;
}

// ---- thread-block cluster primitives: the planner of a large batch runs on a cluster of PLAN_CLUSTER CTAs that exchange scan
// carries and the per-domain tables through distributed shared memory -----------------------------------------------------
__device__ __forceinline__ unsigned cl_rank() { unsigned r; asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r)); return r; }
__device__ __forceinline__ unsigned cl_size() { unsigned r; asm volatile("mov.u32 %0, %%cluster_nctarank;" : "=r"(r)); return r; }
__device__ __forceinline__ void cl_sync_all(unsigned C) {          // every thread of every CTA; release / acquire at cluster scope
    if (C > 1) {
        asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory");
        asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory");
    } else {
        __syncthreads();
    }
}
__device__ __forceinline__ uint32_t cl_map(const void *p, unsigned rank) {   // shared::cluster address of my variable p in CTA `rank`
    uint32_t r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(smem_u32(p)), "r"(rank));
    return r;
}
__device__ __forceinline__ unsigned cl_ld(uint32_t a) { unsigned v; asm volatile("ld.shared::cluster.u32 %0, [%1];" : "=r"(v) : "r"(a) : "memory"); return v; }
__device__ __forceinline__ unsigned long long cl_ld64(uint32_t a) { unsigned long long v; asm volatile("ld.shared::cluster.u64 %0, [%1];" : "=l"(v) : "r"(a) : "memory"); return v; }
__device__ __forceinline__ void cl_red_max(uint32_t a, unsigned v) { asm volatile("red.relaxed.cluster.shared::cluster.max.u32 [%0], %1;" ::"r"(a), "r"(v) : "memory"); }
__device__ __forceinline__ void cl_st(uint32_t a, unsigned v) { asm volatile("st.shared::cluster.u32 [%0], %1;" ::"r"(a), "r"(v) : "memory"); }

#ifndef PLAN_CLUSTER
#define PLAN_CLUSTER 16              // CTAs of the large-batch planner (non-portable cluster size; 8 where 16 cannot be scheduled)
#endif
#define PLAN_CHUNK PLAN_THREADS                  // ops per CTA and super-chunk at full size (the kernel's chunk is blockDim.x)
static_assert(PLAN_CHUNK == PLAN_CHUNK_OPS, "the host planner cuts runs of AMOs / waits where the device planner's chunks end");
// -DSHMEMG_PLAN_TRACE: phase timestamps (%globaltimer, ns) of the planner in the header's spare words hdr->pad3[k]
#ifdef SHMEMG_PLAN_TRACE
#define PTRACE(k) do { if (rank == 0 && tid == 0) { unsigned long long t_; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t_)); a.hdr->pad3[k] = t_; } } while (0)
#else
#define PTRACE(k) do { } while (0)
#endif
// compact per-op key of the keyed pass: domain (bits 0-15), real, wait, counted, has-a-domain
#define KEY_REAL 0x10000u
#define KEY_WAIT 0x20000u
#define KEY_CNT 0x40000u
#define KEY_DOM 0x80000u

struct PlanShared {
    S4 ws[32];
    S4 xtA[PLAN_CLUSTER], xtB[PLAN_CLUSTER];     // block totals of the two scans of a super-chunk, one per cluster rank
    unsigned long long p_bad, p_bulk, f_bad, f_bulk;   // p_: this CTA's partial; f_: reduced over the cluster
    unsigned p_lall, p_mb, p_keyed, p_ptiles, f_lall, f_mb, f_keyed, f_ptiles;
    unsigned all_total;                          // (rank 0) real ops before the last BARRIER_ALL a real op follows
    unsigned dep[PLAN_CHUNK];                    // per-domain thresholds of this CTA's ops of the super-chunk (written by rank 0)
    unsigned char cls[PLAN_CHUNK + 1];           // class of each op of the chunk (1 AMO, 2 wait) | 0x80 = starts a stretch
    unsigned short send[PLAN_CHUNK];             // send[first thread of a stretch] = its last thread (written by that one)
};

// One planner CTA per PLAN_CHUNK ops of a super-chunk (C * PLAN_CHUNK ops); C = cluster size (1 for small batches).
// CL: launched as a thread-block cluster (large batches).  The single-CTA instantiation carries none of the cluster code: the
// planner of a small batch is bound by instruction fetch (cold code in every launch), so its code path is kept short.
// MAXT: upper bound of the CTA size.  A batch of up to 256 ops runs the <false, 256> instantiation, whose register budget is
// not the 64 of a 1024-thread CTA (no spills).
template <bool CL, int MAXT>
__global__ void __launch_bounds__(MAXT, 1) k_plan_batch(const PlanArgs a) {
    extern __shared__ unsigned dsm[];                 // 6 tables of ndom entries, then (rank 0) C * PLAN_CHUNK compact keys
    __shared__ PlanShared sh;
    const unsigned nd = a.ndom;
    unsigned *pL = dsm, *pLnw = dsm + nd, *pM = dsm + 2 * nd;        // partial maxima of this CTA (index + 1; 0 = none)
    unsigned *fL = dsm + 3 * nd, *fLnw = dsm + 4 * nd, *fM = dsm + 5 * nd;   // reduced over the cluster
    unsigned *issued = pL, *thresh = pLnw, *wrun = fL;               // (rank 0, keyed pass) reuse tables that are dead by then
    unsigned *ckey = dsm + 6 * nd;
    const unsigned tid = threadIdx.x, C = CL ? cl_size() : 1u, rank = CL ? cl_rank() : 0u;
    const unsigned NT = blockDim.x;                   // = ops per CTA and super-chunk: PLAN_THREADS, or fewer for a batch of fewer ops
    const unsigned long long n = a.nops, SC = (unsigned long long)C * NT;
    const bool single = n <= SC;                      // one super-chunk: every op stays in its thread's registers
    // the executor may be set up now: it waits (griddepcontrol.wait) until this grid has finished
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    PTRACE(0);
    // Cluster path, one super-chunk: this CTA's descriptors (up to 64 KiB) come in with ONE bulk copy (cp.async.bulk, counted
    // on an mbarrier) while the tables are being zeroed.  A thread that loads its own 64-byte record from global memory makes
    // every warp-level load touch 16 cache lines: 5.2 us for 1024 threads, whether or not the descriptors are in L2.
    __shared__ uint64_t opbar;
    const bool staged = CL && single;
    shmemg_op_t *const ostage = reinterpret_cast<shmemg_op_t *>(dsm + 6 * nd + (size_t)C * PLAN_CHUNK);
    // The planner is itself a programmatic dependent of the kernel before it (an executor releases its dependents at entry):
    // it is resident and has fetched its code while that kernel still runs, and touches nothing -- neither the descriptors,
    // which that kernel may have written, nor the workspace, which a preceding executor still reads -- before this wait.
    asm volatile("griddepcontrol.wait;" ::: "memory");
    if (staged && tid == 0) {
        mbar_init(&opbar, 1);
        mbar_init_fence();
        const unsigned long long first = (unsigned long long)rank * NT;
        const unsigned cnt = first < n ? (unsigned)(n - first < NT ? n - first : NT) : 0u;
        mbar_arrive_expect_tx(&opbar, cnt * (unsigned)sizeof(shmemg_op_t));
        if (cnt) bulk_g2s(ostage, a.ops + first, cnt * (unsigned)sizeof(shmemg_op_t), &opbar);
    }
    for (unsigned d = tid; d < 6 * nd; d += NT) dsm[d] = 0;
    if (tid == 0) { sh.p_bad = ~0ull; sh.p_bulk = 0; sh.p_lall = 0; sh.p_mb = 0; sh.p_keyed = 0; sh.p_ptiles = 0; sh.all_total = 0; }
    __syncthreads();
    if (staged) mbar_wait(&opbar, 0);

    // ======== sweep 1: validate; maxima per domain; totals =====================================================================
    shmemg_op_t keep = {};
    {
        unsigned long long bulk = 0;
        unsigned pt = 0;
        // same-address shared-memory atomics serialise (4096 ops of 64 PEs: 7 us of this sweep), so every warp combines first:
        // ops of one domain are grouped with match.any and the group's HIGHEST lane (the largest op index) updates the table
        unsigned lall_t = 0;
        const unsigned lane = tid & 31;
        for (unsigned long long c0 = (unsigned long long)rank * NT; c0 < n; c0 += SC) {      // uniform trip count per CTA
            const unsigned long long i = c0 + tid;
            const bool have = i < n;
            shmemg_op_t o = {};
            if (have) o = staged ? ostage[tid] : d_ld_op(a.ops + i);
            if (single) keep = o;
            const int rc = have ? d_validate(a, o) : 0;
            if (rc) atomicMin(&sh.p_bad, (i << 8) | (unsigned long long)(-rc));
            const bool real = have && !rc && !d_marker(o.opcode);
            const unsigned dom = real ? (unsigned)o.initiator_pe + (unsigned)o.ctx * (unsigned)a.npes : 0u;
            unsigned grp = 1u << lane, nw = (real && o.opcode != SHMEMG_OP_SIGNAL_WAIT_UNTIL) ? grp : 0u;
            if (CL) {                                   // (a small batch on a few warps: plain atomics are cheaper than the match)
                grp = __match_any_sync(FULLM, real ? dom : 0x80000000u | lane);
                nw = __ballot_sync(FULLM, real && o.opcode != SHMEMG_OP_SIGNAL_WAIT_UNTIL);
            }
            if (real) {
                if (lane == 31u - (unsigned)__clz((int)grp)) atomicMax(&pL[dom], (unsigned)i + 1u);
                const unsigned g2 = grp & nw;
                if (g2 && lane == 31u - (unsigned)__clz((int)g2)) atomicMax(&pLnw[dom], (unsigned)i + 1u);
                lall_t = (unsigned)i + 1u;
                if (d_copy(o.opcode)) { bulk += o.nbytes; pt += (unsigned)((o.nbytes + SHMEMG_TMA_TILE - 1) / SHMEMG_TMA_TILE); }
            }
        }
        lall_t = __reduce_max_sync(FULLM, lall_t);
        if (lane == 0 && lall_t) atomicMax(&sh.p_lall, lall_t);
        for (int o = 16; o; o >>= 1) { bulk += __shfl_xor_sync(FULLM, bulk, o); pt += __shfl_xor_sync(FULLM, pt, o); }
        if ((tid & 31) == 0 && bulk) { atomicAdd(&sh.p_bulk, bulk); atomicAdd(&sh.p_ptiles, pt); }
    }
    PTRACE(1);
    cl_sync_all(C);
    // last real op / last non-wait real op of every domain, over the cluster: every CTA PUSHES its non-zero partial maxima into
    // every CTA's table with fire-and-forget remote atomics (a pull costs one DSMEM round trip per (domain, CTA) pair and most
    // pairs are empty: 13 us for 512 domains x 16 CTAs); the cluster barrier below makes them visible
    for (unsigned d = tid; d < nd; d += NT) {                        // one domain per thread; most domains are empty
        const unsigned m1 = pL[d], m2 = pLnw[d];
        if (!(m1 | m2)) continue;
        if (C > 1) {
            for (unsigned r = 0; r < C; ++r) {
                if (m1) cl_red_max(cl_map(&fL[d], r), m1);
                if (m2) cl_red_max(cl_map(&fLnw[d], r), m2);
            }
        } else {
            fL[d] = m1;
            fLnw[d] = m2;
        }
    }
    if (tid < 32) {                                    // lane r reads CTA r's partials (one DSMEM round trip), the warp combines
        unsigned long long bad = ~0ull, bulk = 0;
        unsigned lall = 0, pt = 0;
        if (tid < C) {
            if (C > 1) {
                bad = cl_ld64(cl_map(&sh.p_bad, tid)); bulk = cl_ld64(cl_map(&sh.p_bulk, tid));
                lall = cl_ld(cl_map(&sh.p_lall, tid)); pt = cl_ld(cl_map(&sh.p_ptiles, tid));
            } else {
                bad = sh.p_bad; bulk = sh.p_bulk; lall = sh.p_lall; pt = sh.p_ptiles;
            }
        }
        for (int o = 16; o; o >>= 1) {
            const unsigned long long b2 = __shfl_xor_sync(FULLM, bad, o);
            bad = b2 < bad ? b2 : bad;
            bulk += __shfl_xor_sync(FULLM, bulk, o);
            lall = max(lall, __shfl_xor_sync(FULLM, lall, o));
            pt += __shfl_xor_sync(FULLM, pt, o);
        }
        if (tid == 0) { sh.f_bad = bad; sh.f_bulk = bulk; sh.f_lall = lall; sh.f_ptiles = pt; }
    }
    cl_sync_all(C);                                    // the pushed maxima have landed in every CTA's tables
    if (sh.f_bad != ~0ull) {                           // a bad descriptor: nothing is executed (shmemg_batch_status reports it)
        if (rank == 0 && tid == 0) {
            a.hdr->ntiles = 0; a.hdr->nunits = 0; a.hdr->npes = nd; a.hdr->trace_on = 0; a.hdr->ticket = 0; a.hdr->all_total = 0;
            a.hdr->stage_bytes = 16384; a.hdr->nstages = 2;
            a.hdr->status = -(int)(sh.f_bad & 0xff); a.hdr->bad_index = sh.f_bad >> 8;
        }
        cl_sync_all(C);                                // nobody leaves while its shared memory may still be read
        return;
    }
    // the last marker of every domain that a later op follows (FENCE / QUIET: any real op; wait: an op other than a wait), the
    // last BARRIER_ALL that a real op follows
    for (unsigned long long c0 = (unsigned long long)rank * NT; c0 < n; c0 += SC) {
        const unsigned long long i = c0 + tid;
        if (i >= n) continue;
        unsigned opc, ctx; int ini;
        if (single) { opc = keep.opcode; ctx = keep.ctx; ini = keep.initiator_pe; } else d_ld_head(a.ops + i, opc, ctx, ini);
        if (opc == SHMEMG_OP_BARRIER_ALL) { if ((unsigned)i + 1u < sh.f_lall) atomicMax(&sh.p_mb, (unsigned)i + 1u); continue; }
        const unsigned dom = (unsigned)ini + ctx * (unsigned)a.npes;
        if (opc == SHMEMG_OP_FENCE || opc == SHMEMG_OP_QUIET) { if ((unsigned)i + 1u < fL[dom]) { atomicMax(&pM[dom], (unsigned)i + 1u); sh.p_keyed = 1; } }
        else if (opc == SHMEMG_OP_SIGNAL_WAIT_UNTIL) { if ((unsigned)i + 1u < fLnw[dom]) { atomicMax(&pM[dom], (unsigned)i + 1u); sh.p_keyed = 1; } }
    }
    cl_sync_all(C);
    for (unsigned d = tid; d < nd; d += NT) {
        const unsigned m = pM[d];
        if (!m) continue;
        if (C > 1) { for (unsigned r = 0; r < C; ++r) cl_red_max(cl_map(&fM[d], r), m); }
        else fM[d] = m;
    }
    if (tid < 32) {
        unsigned mb = 0, k = 0;
        if (tid < C) {
            if (C > 1) { mb = cl_ld(cl_map(&sh.p_mb, tid)); k = cl_ld(cl_map(&sh.p_keyed, tid)); }
            else { mb = sh.p_mb; k = sh.p_keyed; }
        }
        mb = __reduce_max_sync(FULLM, mb);
        k = __reduce_or_sync(FULLM, k);
        if (tid == 0) { sh.f_mb = mb; sh.f_keyed = k; }
    }
    cl_sync_all(C);                                    // the partial tables are dead from here on
    PTRACE(2);
    const unsigned MBp = sh.f_mb;                      // real op i is counted for barriers iff i + 1 < MBp
    const bool keyed = sh.f_keyed != 0;
    const unsigned total_ptiles = sh.f_ptiles;
    unsigned base_seg;
    {
        const unsigned per_sm = (total_ptiles + (unsigned)a.sm_count - 1u) / (unsigned)a.sm_count;
        base_seg = per_sm >= SEG_TILES_MAX ? SEG_TILES_MAX : (per_sm < 1u ? 1u : per_sm);
    }
    const unsigned tail_tiles = (unsigned)a.sm_count * 8u;       // as seg_tiles_per_op (batch.cu): 64 KiB segments in the last 37 MB
    if (keyed && rank == 0) for (unsigned d = tid; d < nd; d += NT) { issued[d] = 0; thresh[d] = 0; wrun[d] = 0; }

    // ======== sweep 2: one super-chunk at a time: scans, per-domain thresholds, records ==========================================
    S4 carryA = {0, 0, 0, 0}, carryB = {0, 0, 0, 0};
    for (unsigned long long s0 = 0; s0 < n; s0 += SC) {
        const unsigned long long i = s0 + (unsigned long long)rank * NT + tid;
        const bool have = i < n;
        shmemg_op_t o = {};
        if (have) o = single ? keep : d_ld_op(a.ops + i);
        const unsigned opc = have ? o.opcode : (unsigned)SHMEMG_OP_BARRIER_ALL;
        const bool real = have && !d_marker(opc), copy = have && d_copy(opc);
        const unsigned cl = have ? d_class(opc) : 0u;
        const unsigned dom = (real || opc == SHMEMG_OP_FENCE || opc == SHMEMG_OP_QUIET) ? (unsigned)o.initiator_pe + (unsigned)o.ctx * (unsigned)a.npes : 0u;
        // ---- A: planner tiles / real ops / AMO+wait records (prefix sums), stretch starts (prefix maximum) ----
        S4 v = {0, 0, 0, 0};
        if (copy) v.a = (unsigned)((o.nbytes + SHMEMG_TMA_TILE - 1) / SHMEMG_TMA_TILE);
        v.b = real ? 1u : 0u;
        v.c = cl ? 1u : 0u;
        sh.cls[tid] = (unsigned char)cl;
        __syncthreads();
        if (cl) {                                       // a run of AMOs / waits never crosses a chunk boundary
            const unsigned pcl = tid > 0 ? (sh.cls[tid - 1] & 0x7fu) : 0u;      // the neighbour's class (its flag bit may or may not be set yet)
            if (pcl != cl) { v.m = (unsigned)i + 1u; sh.cls[tid] = (unsigned char)(cl | 0x80u); }
        }
        S4 tot;
        S4 inc = block_scan(v, sh.ws, tot);
        if (C > 1 && tid < C) {                         // my total to every CTA of the cluster
            S4 *dst = &sh.xtA[rank];
            const uint32_t ra = cl_map(dst, tid);
            cl_st(ra, tot.a); cl_st(ra + 4, tot.b); cl_st(ra + 8, tot.c); cl_st(ra + 12, tot.m);
        }
        cl_sync_all(C);
        {
            S4 pre = carryA, all = carryA;
            if constexpr (CL) { for (unsigned r = 0; r < C; ++r) { if (r < rank) pre = s4_comb(pre, sh.xtA[r]); all = s4_comb(all, sh.xtA[r]); } }
            else all = s4_comb(all, tot);
            inc = s4_comb(pre, inc);
            carryA = all;
        }
        if (s0 == 0) PTRACE(3);
        const unsigned unit = inc.b - v.b, auxi = inc.c - v.c, sstart = inc.m ? inc.m - 1u : 0u;
        if (have && (unsigned)i + 1u == MBp) { if (C > 1) cl_st(cl_map(&sh.all_total, 0), unit); else sh.all_total = unit; }
        // the last op of a stretch of AMOs / waits tells the stretch's first thread where it ends (read behind the next scan)
        if (cl && (tid + 1 == NT || sh.cls[tid + 1] != (unsigned char)cl)) sh.send[sstart - ((unsigned)i - tid)] = (unsigned short)tid;
        // ---- B: tile records per op -> first tile index; unit count at the latest BARRIER_ALL -> barrier threshold ----
        unsigned seg = 0, ntile = 0;
        unsigned long long dst = 0, src = 0;
        Cut cut = {0, 0, 0, 0, 0, 0};
        S4 v2 = {0, 0, 0, 0};
        if (copy) {
            seg = base_seg;
            if (base_seg == SEG_TILES_MAX && total_ptiles - inc.a < tail_tiles) seg = 2u;
            d_endpoints(a, o, dst, src);
            cut = d_cut(dst, src, o.nbytes, seg);
            ntile = cut.np;
        } else if (cl) {
            ntile = ((unsigned)i - sstart) % AMO_RUN_MAX == 0 ? 1u : 0u;
        } else if (have && opc == SHMEMG_OP_BARRIER_ALL && (unsigned)i + 1u <= MBp) {
            v2.m = unit;                                // real ops before this barrier: all of them are counted
        }
        v2.a = ntile;
        S4 inc2 = block_scan(v2, sh.ws, tot);
        if (C > 1 && tid < C) {
            S4 *d2 = &sh.xtB[rank];
            const uint32_t ra = cl_map(d2, tid);
            cl_st(ra, tot.a); cl_st(ra + 4, tot.b); cl_st(ra + 8, tot.c); cl_st(ra + 12, tot.m);
        }
        // ---- K (first half): compact keys of the super-chunk to rank 0 ----
        const bool counted = real && (unsigned)i + 1u <= fM[dom];
        if (keyed) {
            const bool has_dom = have && opc != SHMEMG_OP_BARRIER_ALL;
            const unsigned key = has_dom ? (KEY_DOM | dom | (real ? KEY_REAL : 0u) | (opc == SHMEMG_OP_SIGNAL_WAIT_UNTIL ? KEY_WAIT : 0u) | (counted ? KEY_CNT : 0u)) : 0u;
            if (C > 1) cl_st(cl_map(&ckey[rank * NT + tid], 0), key); else ckey[tid] = key;
        }
        cl_sync_all(C);
        {
            S4 pre = carryB, all = carryB;
            if constexpr (CL) { for (unsigned r = 0; r < C; ++r) { if (r < rank) pre = s4_comb(pre, sh.xtB[r]); all = s4_comb(all, sh.xtB[r]); } }
            else all = s4_comb(all, tot);
            inc2 = s4_comb(pre, inc2);
            carryB = all;
        }
        const unsigned tile0 = inc2.a - v2.a, dep_all = real ? inc2.m : 0u;
        if (s0 == 0) PTRACE(4);
        // ---- K (second half): per-domain thresholds = keyed prefix count; one warp of rank 0 walks the super-chunk ----
        unsigned dep_pe = 0;
        if (keyed) {
            if (rank == 0 && tid < 32) {
                const unsigned lane = tid, lt_mask = (1u << lane) - 1u, le_mask = lt_mask | (1u << lane);
                const unsigned long long left = n - s0;
                const unsigned cnt = (unsigned)(left < SC ? left : SC);
                for (unsigned e0 = 0; e0 < cnt; e0 += 32) {
                    const unsigned e = e0 + lane;
                    const unsigned key = e < cnt ? ckey[e] : 0u;
                    const bool has_dom = key & KEY_DOM, kreal = key & KEY_REAL, iswait = key & KEY_WAIT;
                    const unsigned d = key & 0xffffu;
                    const unsigned same = __match_any_sync(FULLM, has_dom ? d : 0x80000000u | lane);    // the others group with nobody
                    const unsigned cntmask = __ballot_sync(FULLM, (key & KEY_CNT) != 0), waitmask = __ballot_sync(FULLM, has_dom && iswait);
                    const unsigned lt = same & lt_mask;
                    const unsigned Cd = (has_dom ? issued[d] : 0u) + (unsigned)__popc(lt & cntmask);      // counted ops of the domain before this op
                    const bool prev_wait = lt ? ((waitmask >> (31 - __clz((int)lt))) & 1u) != 0 : (has_dom && wrun[d] != 0);
                    const bool boundary = has_dom && (!kreal || (!iswait && prev_wait));    // FENCE / QUIET, or first non-wait op behind waits
                    const unsigned bmask = __ballot_sync(FULLM, boundary);
                    const unsigned bm = same & le_mask & bmask;
                    const unsigned th_b = __shfl_sync(FULLM, Cd, bm ? 31 - __clz((int)bm) : (int)lane);
                    const unsigned th = bm ? th_b : (has_dom ? thresh[d] : 0u);
                    if (e < cnt) { if (C > 1) cl_st(cl_map(&sh.dep[e % NT], e / NT), th); else sh.dep[e] = th; }
                    __syncwarp();
                    if (has_dom && lane == (unsigned)(31 - __clz((int)same))) {           // last op of the domain in this step
                        issued[d] += (unsigned)__popc(same & cntmask);
                        thresh[d] = th;
                        wrun[d] = iswait ? 1u : 0u;
                    }
                    __syncwarp();
                }
            }
            cl_sync_all(C);
            dep_pe = real ? sh.dep[tid] : 0u;
        }
        // ---- E: the records ----
        if (s0 == 0) PTRACE(5);
        if (real) {
            const unsigned flags = (counted ? TF_CNT_PE : 0u) | ((unsigned)i + 1u < MBp ? TF_CNT_ALL : 0u);
            a.arrive[unit] = 0;
            if (cl) {
                AuxRec r = {};
                r.value = o.value;
                r.initiator = dom; r.dep_pe = dep_pe; r.dep_all = dep_all; r.pe_total = 0;
                if (cl == 1) {
                    r.word = (unsigned long long)(a.base + (size_t)o.target_pe * a.stride + o.rem_off);
                    r.fetch = o.opcode == SHMEMG_OP_ATOMIC_ADD ? 0ull : (unsigned long long)(a.base + (size_t)o.initiator_pe * a.stride + o.loc_off);
                    r.cond = o.cond;
                    r.kind = o.opcode | flags;
                } else {
                    r.word = (unsigned long long)(a.base + (size_t)o.initiator_pe * a.stride + o.loc_off);
                    r.kind = SHMEMG_OP_SIGNAL_WAIT_UNTIL | ((unsigned)o.cmp << 8) | flags;
                }
                d_st_rec(a.aux + auxi, r);
                if (ntile && tile0 < a.cap_tiles) {       // first op of a run: its length = the stretch up to AMO_RUN_MAX ops
                    const unsigned left = (unsigned)sh.send[sstart - ((unsigned)i - tid)] - tid + 1u;     // ops of the stretch from here on
                    const unsigned len = left < AMO_RUN_MAX ? left : AMO_RUN_MAX;
                    TileRec t = {};
                    t.kind = cl == 1 ? T_AMO : T_WAIT; t.nbytes = len; t.nt = 1; t.op = unit;
                    t.src = (unsigned long long)(a.aux + auxi);
                    d_st_rec(a.tiles + tile0, t);
                }
            } else {
                unsigned f = flags | ((dep_pe | dep_all) ? TF_DEPS : 0u);
                unsigned long long sig = 0;
                if (o.opcode == SHMEMG_OP_PUT_SIGNAL) {
                    f |= TF_SIGNAL | ((unsigned)o.sig_op << 8);
                    sig = (unsigned long long)(a.base + (size_t)o.target_pe * a.stride + o.sig_off);
                }
                d_emit_cut(cut, o.nbytes, [&](unsigned p, unsigned kind, unsigned long long off, unsigned len) {
                    if (tile0 + p >= a.cap_tiles) return;
                    TileRec t;
                    t.dst = dst + off; t.src = src + off; t.sig = sig; t.value = o.value;
                    t.nbytes = len; t.kind = kind | f; t.op = unit; t.nt = ntile;
                    t.initiator = dom; t.dep_pe = dep_pe; t.dep_all = dep_all; t.pe_total = 0;
                    d_st_rec(a.tiles + tile0 + p, t);
                });
            }
        }
        __syncthreads();                                // sh.cls / sh.dep are rewritten by the next super-chunk
    }
    // ======== header; the counters of a one-call plan start at zero in every call ================================================
    PTRACE(6);
    if (rank == 0) {
        for (unsigned d = tid; d <= nd; d += NT) a.done[d] = 0;
        if (tid == 0) {
            const unsigned ntiles = carryB.a;
            const bool fits = ntiles <= a.cap_tiles;
            const bool small = sh.f_bulk <= (unsigned long long)EXEC_SMALL_PER_SM * (unsigned long long)a.sm_count;
            a.hdr->ntiles = fits ? ntiles : 0u; a.hdr->nunits = carryA.b; a.hdr->npes = nd; a.hdr->trace_on = 0;
            a.hdr->ticket = 0; a.hdr->all_total = sh.all_total;
            a.hdr->tiles_off = a.tiles_off; a.hdr->aux_off = a.aux_off; a.hdr->done_off = a.done_off; a.hdr->arrive_off = a.arrive_off;
            a.hdr->trace_off = 0;
            a.hdr->stage_bytes = small ? 16384u : 32768u; a.hdr->nstages = small ? 12u : 7u;
            a.hdr->status = fits ? SHMEMG_OK : SHMEMG_ERR_NOMEM; a.hdr->bad_index = fits ? 0ull : (unsigned long long)ntiles;
        }
    }
    cl_sync_all(C);                                    // nobody leaves while its shared memory may still be written or read
}

// ---------------------------------------------------------------------------------------------------------
// host
// ---------------------------------------------------------------------------------------------------------
struct WorkLayout { size_t aux_off, done_off, arrive_off, tiles_off; };
static size_t up256(size_t x) { return (x + 255) / 256 * 256; }
static WorkLayout work_layout(const shmemg_world *w, size_t nops) {
    WorkLayout l;
    l.aux_off = sizeof(PlanHeader);
    l.done_off = l.aux_off + up256(nops * sizeof(AuxRec));
    l.arrive_off = l.done_off + up256(((size_t)SHMEMG_CTX_MAX * w->npes + 1) * 4);
    l.tiles_off = l.arrive_off + up256(nops * 4);
    return l;
}

extern "C" size_t shmemg_batch_work_bytes(const shmemg_world_t *w, size_t nops, uint64_t payload_bytes) {
    if (!w) return 0;
    // tile records: <= 3 per op (unaligned head, tail, one piece) + one per 16 KiB of payload, and never fewer than one per SM
    const size_t tiles = 3 * nops + (size_t)(payload_bytes / GEN_TILE) + (size_t)w->sm_count + 1;
    return work_layout(w, nops).tiles_off + tiles * sizeof(TileRec);
}

extern "C" int shmemg_enqueue_batch_ws(shmemg_world_t *w, const shmemg_op_t *ops_dev, size_t nops, void *work_dev,
                                       size_t work_bytes, void *stream) {
    if (!w || (!ops_dev && nops) || !work_dev) return SHMEMG_ERR_ARG;
    if (((uintptr_t)work_dev % 256) || ((uintptr_t)ops_dev % 16)) return SHMEMG_ERR_ALIGN;
    if (nops == 0) return SHMEMG_OK;
    if (nops >= 0xfffffff0ull) return SHMEMG_ERR_NOMEM;
    const unsigned ndom = (unsigned)SHMEMG_CTX_MAX * (unsigned)w->npes;
    if (ndom > PLAN_DOM_MAX) return SHMEMG_ERR_ARG;                 // more than 512 PEs: plan on the host (shmemg_batch_create)
    const WorkLayout l = work_layout(w, nops);
    if (work_bytes < l.tiles_off + (size_t)w->sm_count * sizeof(TileRec)) return SHMEMG_ERR_NOMEM;
    size_t cap = (work_bytes - l.tiles_off) / sizeof(TileRec);
    if (cap > 0xffffffffull) cap = 0xffffffffull;
    uint8_t *wk = (uint8_t *)work_dev;
    PlanArgs p;
    p.ops = ops_dev; p.nops = nops;
    p.base = w->base; p.stride = w->stride; p.heap_bytes = w->heap_bytes; p.npes = w->npes; p.sm_count = w->sm_count;
    p.hdr = (PlanHeader *)wk; p.tiles = (TileRec *)(wk + l.tiles_off); p.aux = (AuxRec *)(wk + l.aux_off);
    p.done = (unsigned *)(wk + l.done_off); p.arrive = (unsigned *)(wk + l.arrive_off);
    p.cap_tiles = (unsigned)cap; p.ndom = ndom;
    p.tiles_off = l.tiles_off; p.aux_off = l.aux_off; p.done_off = l.done_off; p.arrive_off = l.arrive_off;
    // a small batch is planned by one CTA (no cluster barriers on its critical path), a large one by a cluster of 16 (or 8)
    if (!w->plan_cluster) {                                      // once per world: can a cluster of PLAN_CLUSTER planner CTAs be scheduled?
        w->plan_cluster = 8;
        if (PLAN_CLUSTER > 8 &&
            cudaFuncSetAttribute(k_plan_batch<true, PLAN_THREADS>, cudaFuncAttributeNonPortableClusterSizeAllowed, 1) == cudaSuccess) {
            cudaLaunchConfig_t q = {};
            q.gridDim = dim3(PLAN_CLUSTER); q.blockDim = dim3(PLAN_THREADS);
            q.dynamicSmemBytes = (size_t)6 * PLAN_DOM_MAX * 4 + (size_t)PLAN_CLUSTER * PLAN_CHUNK * 4 + (size_t)PLAN_CHUNK * sizeof(shmemg_op_t);
            cudaLaunchAttribute qa[1];
            qa[0].id = cudaLaunchAttributeClusterDimension;
            qa[0].val.clusterDim.x = PLAN_CLUSTER; qa[0].val.clusterDim.y = 1; qa[0].val.clusterDim.z = 1;
            q.attrs = qa; q.numAttrs = 1;
            int nclusters = 0;
            cudaFuncSetAttribute(k_plan_batch<true, PLAN_THREADS>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)q.dynamicSmemBytes);
            if (cudaOccupancyMaxActiveClusters(&nclusters, k_plan_batch<true, PLAN_THREADS>, &q) == cudaSuccess && nclusters >= 1)
                w->plan_cluster = PLAN_CLUSTER;
        }
        cudaGetLastError();
    }
    const unsigned C = nops <= 2 * PLAN_CHUNK ? 1u : (unsigned)w->plan_cluster;
    // one thread per op: a batch of fewer than PLAN_CHUNK ops is planned by as many warps as it needs (the planner of a small
    // batch is bound by instruction issue: 96 ops on 32 warps take 12 us, on 3 warps 5 us)
    const unsigned NT = nops >= PLAN_CHUNK ? PLAN_CHUNK : (unsigned)((nops + 31) / 32 * 32);
    const size_t smem = (size_t)6 * ndom * 4 + (size_t)C * PLAN_CHUNK * 4 + (C > 1 ? (size_t)PLAN_CHUNK * sizeof(shmemg_op_t) : 0);
    if (!w->smem_attr_plan) {
        SHMEMG_CUDA(w, cudaFuncSetAttribute(k_plan_batch<true, PLAN_THREADS>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                            (int)((size_t)6 * PLAN_DOM_MAX * 4 + (size_t)PLAN_CLUSTER * PLAN_CHUNK * 4 +
                                                  (size_t)PLAN_CHUNK * sizeof(shmemg_op_t))));
        SHMEMG_CUDA(w, cudaFuncSetAttribute(k_plan_batch<false, PLAN_THREADS>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                            (int)((size_t)6 * PLAN_DOM_MAX * 4 + (size_t)PLAN_CHUNK * 4)));
        SHMEMG_CUDA(w, cudaFuncSetAttribute(k_plan_batch<false, 256>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                            (int)((size_t)6 * PLAN_DOM_MAX * 4 + (size_t)PLAN_CHUNK * 4)));
        w->smem_attr_plan = true;
    }
    cudaStream_t st = (cudaStream_t)stream;
    {
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3(C); cfg.blockDim = dim3(NT); cfg.dynamicSmemBytes = smem; cfg.stream = st;
        cudaLaunchAttribute at[1];
        at[0].id = cudaLaunchAttributeClusterDimension;
        at[0].val.clusterDim.x = C; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
        cudaLaunchAttribute at2[2];
        at2[0] = at[0];
        at2[1].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        at2[1].val.programmaticStreamSerializationAllowed = 1;
        cfg.attrs = at2; cfg.numAttrs = w->dependent_launch ? 2 : 1;
        if (C > 1) SHMEMG_CUDA(w, cudaLaunchKernelEx(&cfg, k_plan_batch<true, PLAN_THREADS>, p));
        else if (NT <= 256) SHMEMG_CUDA(w, cudaLaunchKernelEx(&cfg, k_plan_batch<false, 256>, p));
        else SHMEMG_CUDA(w, cudaLaunchKernelEx(&cfg, k_plan_batch<false, PLAN_THREADS>, p));
    }
    ExecArgs a;
    a.tiles = p.tiles; a.ticket = &p.hdr->ticket; a.done = p.done; a.arrive = p.arrive; a.trace = nullptr;
    a.ntiles = 0; a.npes = ndom; a.all_total = 0; a.stage_bytes = 0; a.nstages = 0;
    a.hdr = p.hdr;
    return shmemg_exec_launch(w, a, (unsigned)w->sm_count, EXEC_SMEM_MAX, st, true);
}

extern "C" int shmemg_enqueue_batch(shmemg_world_t *w, const shmemg_op_t *ops_dev, size_t nops, void *stream) {
    if (!w) return SHMEMG_ERR_ARG;
    return shmemg_enqueue_batch_ws(w, ops_dev, nops, w->arena, SHMEMG_ARENA_BYTES, stream);
}

extern "C" int shmemg_batch_status(shmemg_world_t *w, const void *work_dev, void *stream, int *status, size_t *bad_index) {
    if (!w || !status) return SHMEMG_ERR_ARG;
    const PlanHeader *h = (const PlanHeader *)(work_dev ? work_dev : w->arena);
    struct { int32_t status; uint32_t pad; unsigned long long bad; } v;
    SHMEMG_CUDA(w, cudaMemcpyAsync(&v, &h->status, sizeof(v), cudaMemcpyDeviceToHost, (cudaStream_t)stream));
    SHMEMG_CUDA(w, cudaStreamSynchronize((cudaStream_t)stream));
    *status = v.status;
    if (bad_index) *bad_index = (size_t)v.bad;
    return SHMEMG_OK;
}
