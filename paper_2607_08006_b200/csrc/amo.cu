// amo.cu -- homogeneous AMO batches in structure-of-arrays form.
//
// One grid-stride kernel per call; op i targets the 64-bit word  base + tgt_pe[i]*stride + sym_off + 8*idx[i].
// Non-fetching add uses red.global (fire-and-forget at the L2 atomic unit); fetch-add and compare-swap use
// atom.global and write the fetched value to a dense, coalesced output array.  No ordering exists between
// the ops of one call (non-blocking semantics), which is what lets a warp combine its
// same-address ops into one L2 atomic (SHMEMG_AMO_WARP_AGGREGATE):
//   add        : leader issues red(sum of the group's values);
//   fetch-add  : leader issues atom.add(sum); lane k fetches  base + (sum of values of lower lanes in group),
//                which is the linearisation "group members back to back in lane order";
//   compare-swap with one scalar cond and val != cond: leader issues the CAS; every other member's CAS is
//                linearised right after it and must fail, fetching (old == cond ? leader's val : old).
#include "internal.cuh"

#define AMO_ITEMS 4
#define FULL 0xffffffffu

enum { AMO_ADD = 0, AMO_FADD = 1, AMO_CAS = 2 };

template <int IDXB> struct IdxT;
template <> struct IdxT<4> { typedef unsigned int type; };
template <> struct IdxT<8> { typedef unsigned long long type; };

struct AmoArgs {
    uint8_t *base;
    size_t stride;
    uint64_t sym_off;
    const int *tgt_pe;
    const void *idx;
    const unsigned long long *val;
    unsigned long long val_s;
    const unsigned long long *cond;
    unsigned long long cond_s;
    unsigned long long *fetched;
    size_t n;
    CtlRegion *then_barrier;       // SHMEMG_AMO_THEN_BARRIER: the CTA that finishes last bumps the world's barrier epoch
};

// quiet + barrier_all folded into the end of an AMO kernel: the end of the kernel completes every AMO of the call (quiet for
// every PE) and orders it before everything later on the stream; what a separate barrier launch would add is the epoch bump,
// which the last CTA to finish performs after a GPU-scope fence.
__device__ __forceinline__ void amo_then_barrier(CtlRegion *ctl) {
    if (!ctl) return;
    __syncthreads();
    if (threadIdx.x == 0) {
        __threadfence();
        if (atomicAdd(&ctl->amo_done, 1u) == gridDim.x - 1) {
            ctl->amo_done = 0;
            __threadfence();
            atomicAdd(&ctl->barrier_epoch, 1ull);
        }
    }
}

__device__ __forceinline__ unsigned long long shfl64(unsigned long long v, int lane) {
    return __shfl_sync(FULL, v, lane);
}

template <int IDXB, int OP, bool AGG, bool TEST>
__global__ void __launch_bounds__(256) k_amo(const AmoArgs a) {     // (256, 6) and (256, 8) spill and are slower: 661 / 757 us vs 590 (C4 CAS)
    typedef typename IdxT<IDXB>::type idx_t;
    const idx_t *__restrict__ idx = reinterpret_cast<const idx_t *>(a.idx);
    const int *__restrict__ tgt = a.tgt_pe;
    const unsigned long long *__restrict__ val = a.val;
    const unsigned long long *__restrict__ cond = a.cond;
    const size_t T = (size_t)gridDim.x * blockDim.x;
    const int lane = threadIdx.x & 31;
    // warp-uniform trip count so that the full-mask warp primitives below are legal
    const size_t warp_first = ((size_t)blockIdx.x * blockDim.x + threadIdx.x) - lane;
    for (size_t i0 = warp_first; i0 < a.n; i0 += T * AMO_ITEMS) {
        unsigned long long addr[AMO_ITEMS], v[AMO_ITEMS], c[AMO_ITEMS];
        bool ok[AMO_ITEMS];
#pragma unroll
        for (int k = 0; k < AMO_ITEMS; ++k) {
            const size_t i = i0 + lane + (size_t)k * T;
            ok[k] = i < a.n;
            addr[k] = 0; v[k] = a.val_s; c[k] = a.cond_s;
            if (ok[k]) {
                addr[k] = (unsigned long long)(a.base + (size_t)tgt[i] * a.stride + a.sym_off) + 8ull * (unsigned long long)idx[i];
                if (val) v[k] = val[i];
                if (OP == AMO_CAS && cond) c[k] = cond[i];
            }
        }
        if (OP == AMO_CAS && TEST) {
            // test before compare-swap (scalar cond only): within one call a word that differs from cond can no longer
            // change (every op swaps only cond -> val, val != cond), so a coherent load that sees such a value IS the
            // failed compare-swap, linearised at the load; the L2 atomic is issued only while the word may still be cond.
            unsigned long long cur[AMO_ITEMS];
#pragma unroll
            for (int k = 0; k < AMO_ITEMS; ++k)
                cur[k] = (ok[k] && v[k] != c[k]) ? ld_relaxed_u64(reinterpret_cast<const unsigned long long *>(addr[k])) : c[k];
#pragma unroll
            for (int k = 0; k < AMO_ITEMS; ++k)
                if (cur[k] != c[k]) {
                    a.fetched[i0 + lane + (size_t)k * T] = cur[k];
                    ok[k] = false;
                }
        }
#pragma unroll
        for (int k = 0; k < AMO_ITEMS; ++k) {
            const size_t i = i0 + lane + (size_t)k * T;
            unsigned long long *word = reinterpret_cast<unsigned long long *>(addr[k]);
            if (!AGG) {
                if (!ok[k]) continue;
                if (OP == AMO_ADD) {
                    asm volatile("red.relaxed.gpu.global.add.u64 [%0], %1;" ::"l"(word), "l"(v[k]) : "memory");
                } else if (OP == AMO_FADD) {
                    a.fetched[i] = atomicAdd(word, v[k]);
                } else {
                    a.fetched[i] = atomicCAS(word, c[k], v[k]);
                }
                continue;
            }
            if (TEST && !__any_sync(FULL, ok[k])) continue;       // every lane was resolved by the test load
            // ---- warp aggregation: lanes that may not combine get a key no other lane can have ----
            const bool solo = !ok[k] || (OP == AMO_CAS && (cond != nullptr || v[k] == c[k]));
            const unsigned long long key = solo ? (unsigned long long)lane : addr[k];   // real addresses are >= 2^32
            const unsigned grp = __match_any_sync(FULL, key);
            const int leader = __ffs(grp) - 1;
            if (!__any_sync(FULL, grp & (grp - 1))) {           // every group is a single lane: plain path
                if (ok[k]) {
                    if (OP == AMO_ADD) asm volatile("red.relaxed.gpu.global.add.u64 [%0], %1;" ::"l"(word), "l"(v[k]) : "memory");
                    else if (OP == AMO_FADD) a.fetched[i] = atomicAdd(word, v[k]);
                    else a.fetched[i] = atomicCAS(word, c[k], v[k]);
                }
                continue;
            }
            if (OP == AMO_CAS) {
                unsigned long long old = 0;
                if (ok[k] && lane == leader) old = atomicCAS(word, c[k], v[k]);
                const unsigned long long lold = shfl64(old, leader);
                const unsigned long long lval = shfl64(v[k], leader);
                if (ok[k]) a.fetched[i] = (lane == leader) ? old : (lold == c[k] ? lval : lold);
            } else {
                unsigned long long sum = 0, prefix = 0;
                for (int l = 0; l < 32; ++l) {                   // uniform loop: every lane takes part in the shuffles
                    const unsigned long long vl = shfl64(v[k], l);
                    if ((grp >> l) & 1u) {
                        sum += vl;
                        if (l < lane) prefix += vl;
                    }
                }
                if (OP == AMO_ADD) {
                    if (ok[k] && lane == leader)
                        asm volatile("red.relaxed.gpu.global.add.u64 [%0], %1;" ::"l"(word), "l"(sum) : "memory");
                } else {
                    unsigned long long old = 0;
                    if (ok[k] && lane == leader) old = atomicAdd(word, sum);
                    const unsigned long long lold = shfl64(old, leader);
                    if (ok[k]) a.fetched[i] = lold + prefix;
                }
            }
        }
    }
    amo_then_barrier(a.then_barrier);
}


// ---- compare-swap with test-before-swap, streaming form (SHMEMG_AMO_TEST_BEFORE_SWAP, scalar cond, 32-bit word index) -------
// Within one call a word that differs from cond can no longer change (every op swaps only cond -> val; an op whose val equals
// cond leaves the word as it is), so a load that sees such a value IS the failed compare-swap, linearised at the load.  Most ops
// of a claim-a-slot stream (C4: 2^26 ops on 2^22 slots) end there.  Two consequences shape the kernel:
//   * the test load may be served by L1 (ld.global.ca): L1 starts empty at kernel entry, so a value found there was the word's
//     value at some instant of THIS call; if it differs from cond it is final, and if it is a stale cond the L2 atomic that
//     follows decides.  The hot slots of a skewed stream are then answered by the SM's own L1 instead of queueing at the one
//     L2 slice that owns their line (C4: 558 -> 373 us; with L2-coherent test loads 487 us);
//   * the op's VALUE is read only when the word may still be cond (at most once per slot plus races): the operand stream
//     drops from 24 to 16 bytes per op (tgt_pe 4 + idx 4 read, 8 fetched written), and a 32-bit word index per op in flight
//     keeps the register count at 32.
#define CAS_ITEMS 4
__device__ __forceinline__ unsigned long long ld_ca_u64(const unsigned long long *p) {
    unsigned long long v;
    asm volatile("ld.global.ca.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}
template <int IDXB>
__global__ void __launch_bounds__(256) k_cas_test(const AmoArgs a) {
    typedef typename IdxT<IDXB>::type idx_t;
    const idx_t *__restrict__ idx = reinterpret_cast<const idx_t *>(a.idx);
    const int *__restrict__ tgt = a.tgt_pe;
    const unsigned words_per_pe = (unsigned)(a.stride >> 3), word0 = (unsigned)(a.sym_off >> 3);
    unsigned long long *const slab = reinterpret_cast<unsigned long long *>(a.base);
    const unsigned long long c = a.cond_s;
    const size_t T = (size_t)gridDim.x * blockDim.x;
    for (size_t i0 = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i0 < a.n; i0 += T * CAS_ITEMS) {
        unsigned key[CAS_ITEMS];
        unsigned long long cur[CAS_ITEMS];
#pragma unroll
        for (int k = 0; k < CAS_ITEMS; ++k) {
            const size_t i = i0 + (size_t)k * T;
            key[k] = i < a.n ? (unsigned)tgt[i] * words_per_pe + word0 + (unsigned)idx[i] : 0xffffffffu;
        }
#pragma unroll
        for (int k = 0; k < CAS_ITEMS; ++k) cur[k] = key[k] != 0xffffffffu ? ld_ca_u64(slab + key[k]) : c;
#pragma unroll
        for (int k = 0; k < CAS_ITEMS; ++k) {
            if (key[k] == 0xffffffffu) continue;
            const size_t i = i0 + (size_t)k * T;
            if (cur[k] == c) cur[k] = atomicCAS(slab + key[k], c, a.val ? a.val[i] : a.val_s);
            a.fetched[i] = cur[k];
        }
    }
    amo_then_barrier(a.then_barrier);
}

// ---- hot-set aggregation (SHMEMG_AMO_HOT_AGGREGATE; add / fetch-add with ONE scalar value) -----------------------------
// A skewed op stream (C4: RMAT) is bound by same-line serialisation at the L2 atomic unit: the hottest 128-byte line takes
// 0.71 % of the 2^26 ops and its ops alone last as long as the whole kernel (2.7 ns each), while the atomic units idle
// (profiles/r01d).  Removing the 256 hottest words from the stream brings the plain kernel from 1339 to 721 us.  So:
//   k_hot_sample     HOT_SAMPLES ops of the stream are fetched by 16 co-resident CTAs; each of them then counts the keys of its
//                    sixteenth of a hash table in shared memory and publishes the words seen at least HOT_THRESHOLD times
//                    (at most SHMEMG_HOT_MAX) in the control region (13 us);
//   k_amo_hot_main   k_amo's loop with a two-load shared-memory lookup per op.  Cold ops go straight to L2.  The hot ops of a
//                    CTA are combined: ONE L2 atomic per hot word and CTA (count * val); a hot fetch-add receives
//                    old + rank * val, its rank taken from the word's shared-memory counter.
// Measured on C4 (2^26 fetch-adds, RMAT): 1340 -> 850 us (profiles/r02b_fetch_add.md).  What did NOT work on the way (profiles/r01d): a hash table over ALL
// ops of a chunk (2000 us: barriers behind probe loops); contiguous chunks with per-thread hot bitmasks (1090-1530 us: 38-55
// registers cut the number of L2 atomics in flight, which is what this kernel lives on); a separate fix-up kernel re-reading
// the operands of the hot ops (430 us of 32-byte-sector traffic).
// Linearisation: the hot ops of one CTA execute back to back, in rank order, at the instant of the CTA's L2 atomic on
// that word -- legal because the ops of one call are unordered (PAPER L369 / reading 7), the same argument as for warp
// aggregation.  Which words count as hot only changes the speed, never the result.
#define HOT_SAMPLES 16384
#define HOT_SLOTS_SAMPLE 24576u          // 8-byte {key, count} slots of the sampling table, 1536 (12 KiB of shared memory) per sampling CTA
#define HOT_THRESHOLD 3u
#define HOT_INDEX 4096u                  // per-CTA direct-mapped index of the hot words (8 KiB)
#define HOT_NONE 0xffffu
#define HOT_EMPTY 0xffffffffu

__device__ __forceinline__ unsigned hot_hash(unsigned key, unsigned slots) {
    return (unsigned)(((unsigned long long)(key * 0x9E3779B1u) * slots) >> 32);
}

// HOT_SAMPLES / 1024 = 16 CTAs of 1024 threads, co-resident (cooperative launch).  Every thread fetches ONE sample (one SM alone
// cannot keep 2 x 16384 scattered sector loads in flight: 96 us) and stages its key.  When all CTAs have staged (a monotonic
// arrival counter, the round found from the counter alone as in the in-kernel barrier), every CTA counts the keys that hash
// into ITS sixteenth of the sampling table in its own shared memory and appends the words seen at least HOT_THRESHOLD times to
// the control region: one SM building the whole table spent 25 us on 32 Ki shared-memory atomics and 13 us on the scan
// (43 us per call; 13 us this way).
#define HOT_PART (HOT_SLOTS_SAMPLE / (HOT_SAMPLES / 1024))      // table slots per CTA
template <int IDXB>
__global__ void __launch_bounds__(1024) k_hot_sample(const AmoArgs a, CtlRegion *ctl, unsigned *staged) {
    typedef typename IdxT<IDXB>::type idx_t;
    __shared__ __align__(16) unsigned long long stab[HOT_PART];      // {key (low), count (high)}
    unsigned *tab = reinterpret_cast<unsigned *>(stab);
    __shared__ unsigned s_target;
    const idx_t *__restrict__ idx = reinterpret_cast<const idx_t *>(a.idx);
    const unsigned long long words_per_pe = a.stride >> 3, word0 = a.sym_off >> 3;
    const unsigned nb = gridDim.x;
    {
        const size_t q = (size_t)blockIdx.x * 1024 + threadIdx.x, i = q * (a.n / HOT_SAMPLES);   // n >= 2^20: step >= 64
        staged[q] = (unsigned)((unsigned long long)a.tgt_pe[i] * words_per_pe + word0 + (unsigned long long)idx[i]);
    }
    for (unsigned s = threadIdx.x; s < HOT_PART; s += 1024) stab[s] = (unsigned long long)HOT_EMPTY;
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) {
        // before its own arrival a CTA reads a value in [k*nb, (k+1)*nb) of the k-th call on this world (2^32 is a multiple of nb)
        const unsigned c0 = ld_relaxed_u32(&ctl->hot_done);
        if (blockIdx.x == 0) ctl->hot_n = 0;                          // ordered before this CTA's arrival, which every CTA awaits
        s_target = c0 - c0 % nb + nb;
        red_release_add_u32(&ctl->hot_done, 1u);
        while ((int)(ld_relaxed_u32(&ctl->hot_done) - s_target) < 0) { }
        fence_acquire();
    }
    __syncthreads();
    // every staged key is visible now; mine are those that hash into [blockIdx.x * HOT_PART, (blockIdx.x + 1) * HOT_PART)
    const unsigned lo = blockIdx.x * HOT_PART;
    unsigned keys[HOT_SAMPLES / 1024];
#pragma unroll
    for (unsigned u = 0; u < HOT_SAMPLES / 1024; ++u) keys[u] = ld_relaxed_u32(staged + threadIdx.x + u * 1024);
#pragma unroll
    for (unsigned u = 0; u < HOT_SAMPLES / 1024; ++u) {
        const unsigned key = keys[u];
        unsigned h = hot_hash(key, HOT_SLOTS_SAMPLE) - lo;
        if (h >= HOT_PART) continue;                                  // another CTA's key
        unsigned probes = 0;                                          // about 1024 distinct keys per partition of 1536 slots; a
        for (; probes < HOT_PART; ++probes) {                         // partition that overflows drops the key (speed only)
            const unsigned old = atomicCAS(&tab[2 * h], HOT_EMPTY, key);
            if (old == HOT_EMPTY || old == key) break;
            if (++h == HOT_PART) h = 0;
        }
        if (probes < HOT_PART) atomicAdd(&tab[2 * h + 1], 1u);
    }
    __syncthreads();
    for (unsigned s = threadIdx.x; s < HOT_PART; s += 1024) {
        if (tab[2 * s] != HOT_EMPTY && tab[2 * s + 1] >= HOT_THRESHOLD) {
            const unsigned k = atomicAdd(&ctl->hot_n, 1u);            // may run past SHMEMG_HOT_MAX: the readers clamp
            if (k < SHMEMG_HOT_MAX) ctl->hot_keys[k] = tab[2 * s];
        }
    }
}

// shared-memory lookup of the hot words: direct-mapped index hidx[hash(key)] -> j with hkeys[j] == key.  A hot word whose
// index slot is taken by another one is simply not treated as hot (a few per cent): two loads, no loop.
struct HotTable {
    unsigned short hidx[HOT_INDEX];
    unsigned hkeys[SHMEMG_HOT_MAX];
    __device__ __forceinline__ void build(const CtlRegion *ctl, unsigned tid, unsigned nthr) {
        for (unsigned s = tid; s < HOT_INDEX; s += nthr) hidx[s] = HOT_NONE;
        for (unsigned s = tid; s < SHMEMG_HOT_MAX; s += nthr) hkeys[s] = HOT_EMPTY;
        __syncthreads();
        const unsigned nh = ctl->hot_n < SHMEMG_HOT_MAX ? ctl->hot_n : SHMEMG_HOT_MAX;
        for (unsigned k = tid; k < nh; k += nthr) {
            const unsigned key = ctl->hot_keys[k];
            hkeys[k] = key;
            hidx[hot_hash(key, HOT_INDEX)] = (unsigned short)k;       // racing writers: one wins, the losers stay cold
        }
        __syncthreads();
    }
    __device__ __forceinline__ int lookup(unsigned key) const {       // index of a hot word, or -1
        const unsigned j = hidx[hot_hash(key, HOT_INDEX)] & (SHMEMG_HOT_MAX - 1);
        return hkeys[j] == key ? (int)j : -1;
    }
};

// k_amo's grid-stride loop (whole waves of resident CTAs).  Cold ops go to L2.  Hot ops:
//   add        counted in shared memory; one red per hot word and CTA at the end;
//   fetch-add  appended to the CTA's own list in `lists` (op index + hot-word index, coalesced 8-byte records; when the list
//              is full the op simply goes to L2 like a cold one); its rank is taken from the word's shared-memory counter at
//              once and stored in the record.  After the loop: base = ONE L2 atom.add(word, count * val) per hot word, then
//              one pass over the list: fetched = base + rank * val (a separate rank pass cost 25 us: 910 -> 885 us on C4).
#define HOT_I_BITS 34                    // record = op index (34 bits) | hot-word index (9 bits) << 34 | rank (21 bits) << 43
template <int IDXB, int OP>
__global__ void __launch_bounds__(256, 6) k_amo_hot_main(const AmoArgs a, const CtlRegion *ctl, unsigned long long *lists, unsigned cap) {
    typedef typename IdxT<IDXB>::type idx_t;
    __shared__ HotTable ht;
    __shared__ unsigned long long slot[SHMEMG_HOT_MAX];               // count; after the base atomics: the word's old value
    __shared__ unsigned list_n;
    const idx_t *__restrict__ idx = reinterpret_cast<const idx_t *>(a.idx);
    const int *__restrict__ tgt = a.tgt_pe;
    const unsigned long long words_per_pe = a.stride >> 3, word0 = a.sym_off >> 3;
    unsigned long long *const slab = reinterpret_cast<unsigned long long *>(a.base);
    unsigned long long *const list = lists + (size_t)blockIdx.x * cap;
    for (unsigned s = threadIdx.x; s < SHMEMG_HOT_MAX; s += blockDim.x) slot[s] = 0;
    if (threadIdx.x == 0) list_n = 0;
    ht.build(ctl, threadIdx.x, blockDim.x);
    const size_t T = (size_t)gridDim.x * blockDim.x;
    const int lane = threadIdx.x & 31;
    const size_t warp_first = ((size_t)blockIdx.x * blockDim.x + threadIdx.x) - lane;
    for (size_t i0 = warp_first; i0 < a.n; i0 += T * AMO_ITEMS) {
        unsigned key[AMO_ITEMS];
        int hot[AMO_ITEMS];
#pragma unroll
        for (int k = 0; k < AMO_ITEMS; ++k) {
            const size_t i = i0 + lane + (size_t)k * T;
            key[k] = HOT_EMPTY;
            if (i < a.n) key[k] = (unsigned)((unsigned long long)tgt[i] * words_per_pe + word0 + (unsigned long long)idx[i]);
        }
#pragma unroll
        for (int k = 0; k < AMO_ITEMS; ++k) hot[k] = key[k] == HOT_EMPTY ? -2 : ht.lookup(key[k]);     // -2: no op, -1: cold
        unsigned long long old[AMO_ITEMS];
#pragma unroll
        for (int k = 0; k < AMO_ITEMS; ++k) {                         // the L2 atomics first: everything below overlaps them
            if (hot[k] == -1) {
                if (OP == AMO_ADD) asm volatile("red.relaxed.gpu.global.add.u64 [%0], %1;" ::"l"(slab + key[k]), "l"(a.val_s) : "memory");
                else old[k] = atomicAdd(slab + key[k], a.val_s);
            } else if (OP == AMO_ADD && hot[k] >= 0) {
                atomicAdd(reinterpret_cast<unsigned *>(&slot[hot[k]]), 1u);       // < 2^32 ops per CTA
            }
        }
        if (OP == AMO_FADD) {
#pragma unroll
            for (int k = 0; k < AMO_ITEMS; ++k) {                     // warp-aggregated append to the CTA's list
                const unsigned b = __ballot_sync(FULL, hot[k] >= 0);
                if (b == 0) continue;
                unsigned pos = 0;
                if (lane == __ffs((int)b) - 1) pos = atomicAdd(&list_n, (unsigned)__popc(b));
                pos = __shfl_sync(FULL, pos, __ffs((int)b) - 1) + (unsigned)__popc(b & ((1u << lane) - 1u));
                if (hot[k] >= 0) {
                    if (pos < cap) {                                  // the rank is taken now: no separate rank pass at the end
                        const unsigned rank = atomicAdd(reinterpret_cast<unsigned *>(&slot[hot[k]]), 1u);
                        list[pos] = (unsigned long long)(i0 + lane + (size_t)k * T) | ((unsigned long long)hot[k] << HOT_I_BITS) |
                                    ((unsigned long long)rank << 43);
                    } else {                                          // list full: an ordinary L2 atomic after all
                        old[k] = atomicAdd(slab + key[k], a.val_s);
                        hot[k] = -1;
                    }
                }
            }
        }
        if (OP == AMO_FADD) {
#pragma unroll
            for (int k = 0; k < AMO_ITEMS; ++k)
                if (hot[k] == -1) a.fetched[i0 + lane + (size_t)k * T] = old[k];
        }
    }
    __syncthreads();
    if (OP == AMO_ADD) {
        for (unsigned j = threadIdx.x; j < SHMEMG_HOT_MAX; j += blockDim.x) {
            const unsigned long long c = slot[j];
            if (c) asm volatile("red.relaxed.gpu.global.add.u64 [%0], %1;" ::"l"(slab + ht.hkeys[j]), "l"(c * a.val_s) : "memory");
        }
        amo_then_barrier(a.then_barrier);
        return;
    }
    const unsigned nl = list_n < cap ? list_n : cap;
    const unsigned long long imask = (1ull << HOT_I_BITS) - 1;
    for (unsigned j = threadIdx.x; j < SHMEMG_HOT_MAX; j += blockDim.x) {
        const unsigned long long c = slot[j];
        if (c) slot[j] = atomicAdd(slab + ht.hkeys[j], c * a.val_s);
    }
    __syncthreads();
    for (unsigned e = threadIdx.x; e < nl; e += blockDim.x) {         // records written by this CTA before the first barrier
        const unsigned long long r = list[e];
        a.fetched[r & imask] = slot[(r >> HOT_I_BITS) & (SHMEMG_HOT_MAX - 1)] + (r >> 43) * a.val_s;
    }
    amo_then_barrier(a.then_barrier);
}

// usable when the value is one scalar and every word of the slab has a 32-bit index; small calls keep the plain kernel
static bool hot_agg_ok(const shmemg_world *w, const AmoArgs &a, uint32_t flags) {
    return (flags & SHMEMG_AMO_HOT_AGGREGATE) && a.val == nullptr && (a.stride & 7) == 0 &&
           ((uint64_t)w->npes * a.stride >> 3) < 0xffffffffull && a.n >= ((size_t)1 << 20) && a.n < ((size_t)1 << 33);
}

template <int OP>
static int launch_amo_hot(shmemg_world *w, const AmoArgs &a, int idx_bytes, cudaStream_t st) {
    // whole waves of resident CTAs; every CTA may list up to 1/8 of its ops as hot (what does not fit goes to L2 directly)
    int per_sm = 0;
    if (idx_bytes == 4) cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_amo_hot_main<4, OP>, 256, 0);
    else cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_amo_hot_main<8, OP>, 256, 0);
    if (per_sm < 1) per_sm = 1;
    size_t waves = 8;                                         // measured on C4: 1 wave 970 us, 8 waves 890 us, 32 waves 980 us
#ifdef SHMEMG_EXPERIMENTS
    if (const char *e = getenv("SHMEMG_HOT_WAVES")) waves = (size_t)atoi(e) > 0 ? (size_t)atoi(e) : waves;   // shmemg_amo_scratch_bytes assumes 8
#endif
    const size_t blocks = (size_t)w->sm_count * per_sm * waves;
    const size_t per_cta = (a.n + blocks - 1) / blocks;
    if (per_cta >= ((size_t)1 << 21) * 8 || a.n >= ((size_t)1 << HOT_I_BITS)) return SHMEMG_ERR_NOMEM;   // caller falls back
    unsigned cap = (unsigned)(per_cta / 8 + 32);
    if (cap > (1u << 21)) cap = 1u << 21;                     // the rank field of a hot-op record is 21 bits
    // scratch comes from the caller (shmemg_set_scratch): the library allocates no device memory
    const size_t need = (size_t)HOT_SAMPLES * 4 + (OP == AMO_FADD ? blocks * (size_t)cap * 8 : 0);
    if (!w->scratch || w->scratch_bytes < need) return SHMEMG_ERR_NOMEM;     // caller falls back to the plain kernel
    unsigned long long *lists = OP == AMO_FADD ? (unsigned long long *)((uint8_t *)w->scratch + (size_t)HOT_SAMPLES * 4) : nullptr;
    unsigned *staged = (unsigned *)w->scratch;
    {   // the 16 sampling CTAs wait for one another: cooperative launch (co-resident or refused)
        AmoArgs aa = a;
        CtlRegion *ctl = w->ctl;
        void *args[] = {&aa, &ctl, &staged};
        const void *fn = idx_bytes == 4 ? (const void *)k_hot_sample<4> : (const void *)k_hot_sample<8>;
        if (cudaLaunchCooperativeKernel(fn, dim3(HOT_SAMPLES / 1024), dim3(1024), args, 0, st) != cudaSuccess) {
            cudaGetLastError();
            return SHMEMG_ERR_NOMEM;                            // caller falls back to the plain kernel
        }
    }
    if (idx_bytes == 4) k_amo_hot_main<4, OP><<<(unsigned)blocks, 256, 0, st>>>(a, w->ctl, lists, cap);
    else k_amo_hot_main<8, OP><<<(unsigned)blocks, 256, 0, st>>>(a, w->ctl, lists, cap);
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return shmemg_cuda_fail(w, e, "k_amo_hot");
    return SHMEMG_OK;
}

template <int OP>
static int launch_amo(shmemg_world *w, const AmoArgs &a, int idx_bytes, uint32_t flags, cudaStream_t st) {
    if (a.n == 0) return a.then_barrier ? shmemg_barrier_all_on_stream(w, st) : SHMEMG_OK;
    const int threads = 256;
    // one op per thread until the grid is full (a 65 536-op batch then runs on 256 CTAs instead of 64: its time is the latency
    // of one trip, so it wants every SM), AMO_ITEMS ops per thread and trip beyond that
    size_t blocks = (a.n + (size_t)threads - 1) / (size_t)threads;
    const size_t cap = (size_t)w->sm_count * 8 * 4;        // 8 resident CTAs per SM, ~4 waves worth of grid stride
    if (blocks > cap) blocks = cap;
    const bool agg = flags & SHMEMG_AMO_WARP_AGGREGATE;
    const bool test = OP == AMO_CAS && (flags & SHMEMG_AMO_TEST_BEFORE_SWAP) && a.cond == nullptr;
    if (test && !agg && (a.stride & 7) == 0 && ((uint64_t)w->npes * a.stride >> 3) < 0xffffffffull) {
        // streaming form: every word of the slab has a 32-bit index (slab < 32 GiB)
        if (idx_bytes == 4) k_cas_test<4><<<(unsigned)blocks, threads, 0, st>>>(a);
        else k_cas_test<8><<<(unsigned)blocks, threads, 0, st>>>(a);
        SHMEMG_CUDA(w, cudaGetLastError());
        return SHMEMG_OK;
    }
    if (idx_bytes == 4) {
        if (test) { if (agg) k_amo<4, OP, true, true><<<(unsigned)blocks, threads, 0, st>>>(a);
                    else k_amo<4, OP, false, true><<<(unsigned)blocks, threads, 0, st>>>(a); }
        else if (agg) k_amo<4, OP, true, false><<<(unsigned)blocks, threads, 0, st>>>(a);
        else k_amo<4, OP, false, false><<<(unsigned)blocks, threads, 0, st>>>(a);
    } else {
        if (test) { if (agg) k_amo<8, OP, true, true><<<(unsigned)blocks, threads, 0, st>>>(a);
                    else k_amo<8, OP, false, true><<<(unsigned)blocks, threads, 0, st>>>(a); }
        else if (agg) k_amo<8, OP, true, false><<<(unsigned)blocks, threads, 0, st>>>(a);
        else k_amo<8, OP, false, false><<<(unsigned)blocks, threads, 0, st>>>(a);
    }
    SHMEMG_CUDA(w, cudaGetLastError());
    return SHMEMG_OK;
}

static int check_common(shmemg_world *w, uint64_t sym_off, const int32_t *tgt_pe, const void *elem_idx, int idx_bytes,
                        size_t n) {
    if (!w) return SHMEMG_ERR_ARG;
    if (n && (!tgt_pe || !elem_idx)) return SHMEMG_ERR_ARG;
    if (idx_bytes != 4 && idx_bytes != 8) return SHMEMG_ERR_ARG;
    if (sym_off & 7) return SHMEMG_ERR_ALIGN;
    if (!shmemg_in_range(w, sym_off, 8)) return SHMEMG_ERR_RANGE;
    // tgt_pe[] and elem_idx[] are DEVICE arrays: per-op bounds are the caller's contract (undefined otherwise)
    return SHMEMG_OK;
}

extern "C" int shmemg_atomic_add_batch_on_stream(shmemg_world_t *w, uint64_t sym_off, const int32_t *tgt_pe,
                                                 const void *elem_idx, int idx_bytes, const uint64_t *val,
                                                 uint64_t val_scalar, size_t n, uint32_t flags, void *stream) {
    int rc = check_common(w, sym_off, tgt_pe, elem_idx, idx_bytes, n);
    if (rc) return rc;
    AmoArgs a{w->base, w->stride, sym_off, tgt_pe, elem_idx, (const unsigned long long *)val, val_scalar, nullptr, 0, nullptr, n,
              (flags & SHMEMG_AMO_THEN_BARRIER) ? w->ctl : nullptr};
    w->amo_last_path = 0;
    if (hot_agg_ok(w, a, flags)) {
        rc = launch_amo_hot<AMO_ADD>(w, a, idx_bytes, (cudaStream_t)stream);
        if (rc == SHMEMG_OK) w->amo_last_path = 1;
        if (rc != SHMEMG_ERR_NOMEM) return rc;                 // no (or too small a) scratch buffer: the plain kernel
    }
    return launch_amo<AMO_ADD>(w, a, idx_bytes, flags, (cudaStream_t)stream);
}

extern "C" int shmemg_atomic_fetch_add_batch_on_stream(shmemg_world_t *w, uint64_t sym_off, const int32_t *tgt_pe,
                                                       const void *elem_idx, int idx_bytes, const uint64_t *val,
                                                       uint64_t val_scalar, uint64_t *fetched_out, size_t n,
                                                       uint32_t flags, void *stream) {
    int rc = check_common(w, sym_off, tgt_pe, elem_idx, idx_bytes, n);
    if (rc) return rc;
    if (n && !fetched_out) return SHMEMG_ERR_ARG;
    AmoArgs a{w->base, w->stride, sym_off, tgt_pe, elem_idx, (const unsigned long long *)val, val_scalar, nullptr, 0,
              (unsigned long long *)fetched_out, n, (flags & SHMEMG_AMO_THEN_BARRIER) ? w->ctl : nullptr};
    w->amo_last_path = 0;
    if (hot_agg_ok(w, a, flags)) {
        rc = launch_amo_hot<AMO_FADD>(w, a, idx_bytes, (cudaStream_t)stream);
        if (rc == SHMEMG_OK) w->amo_last_path = 1;
        if (rc != SHMEMG_ERR_NOMEM) return rc;
    }
    return launch_amo<AMO_FADD>(w, a, idx_bytes, flags, (cudaStream_t)stream);
}

extern "C" int shmemg_atomic_compare_swap_batch_on_stream(shmemg_world_t *w, uint64_t sym_off, const int32_t *tgt_pe,
                                                          const void *elem_idx, int idx_bytes, const uint64_t *cond,
                                                          uint64_t cond_scalar, const uint64_t *val,
                                                          uint64_t val_scalar, uint64_t *fetched_out, size_t n,
                                                          uint32_t flags, void *stream) {
    int rc = check_common(w, sym_off, tgt_pe, elem_idx, idx_bytes, n);
    if (rc) return rc;
    if (n && !fetched_out) return SHMEMG_ERR_ARG;
    AmoArgs a{w->base, w->stride, sym_off, tgt_pe, elem_idx, (const unsigned long long *)val, val_scalar,
              (const unsigned long long *)cond, cond_scalar, (unsigned long long *)fetched_out, n,
              (flags & SHMEMG_AMO_THEN_BARRIER) ? w->ctl : nullptr};
    return launch_amo<AMO_CAS>(w, a, idx_bytes, flags, (cudaStream_t)stream);
}


// ---- caller-provided scratch (the library allocates no device memory) -------------------------------------------------------
extern "C" size_t shmemg_amo_scratch_bytes(const shmemg_world_t *w, size_t n) {
    if (!w) return 0;
    // what launch_amo_hot needs for a fetch-add batch of n ops: staged sample keys + the per-CTA hot-op lists
    int per_sm = 0;
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_amo_hot_main<4, AMO_FADD>, 256, 0);
    if (per_sm < 1) per_sm = 1;
    const size_t blocks = (size_t)w->sm_count * per_sm * 8;
    size_t cap = (n + blocks - 1) / blocks / 8 + 32;
    if (cap > ((size_t)1 << 21)) cap = (size_t)1 << 21;
    return (size_t)HOT_SAMPLES * 4 + blocks * cap * 8;
}
extern "C" int shmemg_amo_last_path(const shmemg_world_t *w) { return w ? w->amo_last_path : SHMEMG_ERR_ARG; }
extern "C" int shmemg_set_scratch(shmemg_world_t *w, void *scratch_dev, size_t bytes) {
    if (!w || (!scratch_dev && bytes)) return SHMEMG_ERR_ARG;
    if ((uintptr_t)scratch_dev % 256) return SHMEMG_ERR_ALIGN;
    w->scratch = scratch_dev;
    w->scratch_bytes = scratch_dev ? bytes : 0;
    return SHMEMG_OK;
}

// ---- fetch-add on the library's built-in scratch (shmemg_atomic_fetch_add_batch_static_on_stream) ---------------------------
// For callers that cannot obtain device memory themselves (see include/shmemg.h): the staged sample keys and the per-CTA
// hot-op lists of k_hot_sample / k_amo_hot_main live in this file-scope device array instead of a caller-owned buffer.  The
// array is part of the module image: every GPU that loads libshmemg.so holds these 8 MiB until the process exits.
//
// g_static_scratch is a DEVICE symbol.  Host code must never hand the name itself to a kernel: on the host it stands for a
// shadow object in host memory, so a kernel given `g_static_scratch` faults (or, on a system where the GPU can read host
// memory, quietly works on the wrong bytes).  static_scratch_ptr() asks the runtime for the real device address, once per
// device and with that device current, and the launch below passes THAT pointer.
#include <mutex>

static __device__ __align__(256) unsigned char g_static_scratch[SHMEMG_STATIC_SCRATCH_BYTES];

#define STATIC_MAX_DEVICES 64
static std::mutex g_static_mu;
static unsigned char *g_static_ptr[STATIC_MAX_DEVICES];      // device address of g_static_scratch on device d (0: not asked yet)

static int static_scratch_ptr(shmemg_world *w, unsigned char **out) {
    int cur = -1;
    SHMEMG_CUDA(w, cudaGetDevice(&cur));
    if (cur != w->device || cur < 0 || cur >= STATIC_MAX_DEVICES) {
        w->last_cuda_error = "shmemg_atomic_fetch_add_batch_static_on_stream: the world lives on device " + std::to_string(w->device) +
                             " but device " + std::to_string(cur) + " is current (the built-in scratch is looked up per device)";
        return SHMEMG_ERR_ARG;
    }
    std::lock_guard<std::mutex> lock(g_static_mu);
    if (!g_static_ptr[cur]) {
        void *p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(&p, g_static_scratch);
        if (e != cudaSuccess || !p) return shmemg_cuda_fail(w, e, "cudaGetSymbolAddress(g_static_scratch)");
        g_static_ptr[cur] = (unsigned char *)p;
    }
    *out = g_static_ptr[cur];
    return SHMEMG_OK;
}

extern "C" int shmemg_atomic_fetch_add_batch_static_on_stream(shmemg_world_t *w, uint64_t sym_off, const int32_t *tgt_pe,
                                                              const void *elem_idx, int idx_bytes, uint64_t val_scalar,
                                                              uint64_t *fetched_out, size_t n, uint32_t flags, void *stream,
                                                              int *path_out) {
    if (path_out) *path_out = 0;
    int rc = check_common(w, sym_off, tgt_pe, elem_idx, idx_bytes, n);
    if (rc) return rc;
    if (n && !fetched_out) return SHMEMG_ERR_ARG;
    if (flags & ~(SHMEMG_AMO_THEN_BARRIER | SHMEMG_AMO_HOT_AGGREGATE)) return SHMEMG_ERR_ARG;
    if (n > SHMEMG_STATIC_MAX_OPS) {
        w->last_cuda_error = "shmemg_atomic_fetch_add_batch_static_on_stream: n = " + std::to_string(n) + " ops is more than SHMEMG_STATIC_MAX_OPS = " +
                             std::to_string((size_t)SHMEMG_STATIC_MAX_OPS) + " (the built-in scratch is " +
                             std::to_string((size_t)SHMEMG_STATIC_SCRATCH_BYTES) + " bytes); split the batch or register a buffer with shmemg_set_scratch";
        return SHMEMG_ERR_NOMEM;
    }
    cudaStream_t st = (cudaStream_t)stream;
    AmoArgs a{w->base, w->stride, sym_off, tgt_pe, elem_idx, nullptr, val_scalar, nullptr, 0, (unsigned long long *)fetched_out, n,
              (flags & SHMEMG_AMO_THEN_BARRIER) ? w->ctl : nullptr};
    if (!hot_agg_ok(w, a, SHMEMG_AMO_HOT_AGGREGATE))                        // small call or huge slab: the plain kernel needs no scratch
        return launch_amo<AMO_FADD>(w, a, idx_bytes, 0, st);
    unsigned char *scratch = nullptr;
    rc = static_scratch_ptr(w, &scratch);
    if (rc) return rc;
    // the geometry of launch_amo_hot: 8 waves of resident CTAs, every CTA may list up to 1/8 of its ops (+32) as hot
    int per_sm = 0;
    if (idx_bytes == 4) cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_amo_hot_main<4, AMO_FADD>, 256, 0);
    else cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_amo_hot_main<8, AMO_FADD>, 256, 0);
    if (per_sm < 1) per_sm = 1;
    const size_t blocks = (size_t)w->sm_count * per_sm * 8;
    const unsigned cap = (unsigned)((n + blocks - 1) / blocks / 8 + 32);    // n <= 2^22: far below the 21-bit rank field
    const size_t need = (size_t)HOT_SAMPLES * 4 + blocks * (size_t)cap * 8;
    if (need > SHMEMG_STATIC_SCRATCH_BYTES) {                               // a GPU with far more SMs than the B200 this was sized for
        w->last_cuda_error = "shmemg_atomic_fetch_add_batch_static_on_stream: " + std::to_string(n) + " ops need " + std::to_string(need) +
                             " bytes of scratch on this GPU, the built-in scratch is " + std::to_string((size_t)SHMEMG_STATIC_SCRATCH_BYTES);
        return SHMEMG_ERR_NOMEM;
    }
    // Nothing to clear: k_hot_sample writes all HOT_SAMPLES staged keys before any CTA reads one, and k_amo_hot_main reads only
    // the list records it wrote itself in this launch (their count lives in shared memory), so what the last call left is never read.
    unsigned *staged = (unsigned *)scratch;
    unsigned long long *lists = (unsigned long long *)(scratch + (size_t)HOT_SAMPLES * 4);
    {
        AmoArgs aa = a;
        CtlRegion *ctl = w->ctl;
        void *args[] = {&aa, &ctl, &staged};
        const void *fn = idx_bytes == 4 ? (const void *)k_hot_sample<4> : (const void *)k_hot_sample<8>;
        if (cudaLaunchCooperativeKernel(fn, dim3(HOT_SAMPLES / 1024), dim3(1024), args, 0, st) != cudaSuccess) {
            cudaGetLastError();                                             // the sampling CTAs cannot be co-resident here
            return launch_amo<AMO_FADD>(w, a, idx_bytes, 0, st);
        }
    }
    if (idx_bytes == 4) k_amo_hot_main<4, AMO_FADD><<<(unsigned)blocks, 256, 0, st>>>(a, w->ctl, lists, cap);
    else k_amo_hot_main<8, AMO_FADD><<<(unsigned)blocks, 256, 0, st>>>(a, w->ctl, lists, cap);
    SHMEMG_CUDA(w, cudaGetLastError());
    if (path_out) *path_out = 1;
    return SHMEMG_OK;
}
