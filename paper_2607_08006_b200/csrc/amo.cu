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
};

__device__ __forceinline__ unsigned long long shfl64(unsigned long long v, int lane) {
    return __shfl_sync(FULL, v, lane);
}

template <int IDXB, int OP, bool AGG, bool TEST>
__global__ void __launch_bounds__(256) k_amo(const AmoArgs a) {
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
}

template <int OP>
static int launch_amo(shmemg_world *w, const AmoArgs &a, int idx_bytes, uint32_t flags, cudaStream_t st) {
    if (a.n == 0) return SHMEMG_OK;
    const int threads = 256;
    size_t blocks = (a.n + (size_t)threads * AMO_ITEMS - 1) / ((size_t)threads * AMO_ITEMS);
    const size_t cap = (size_t)w->sm_count * 8 * 4;        // 8 resident CTAs per SM, ~4 waves worth of grid stride
    if (blocks > cap) blocks = cap;
    const bool agg = flags & SHMEMG_AMO_WARP_AGGREGATE;
    const bool test = OP == AMO_CAS && (flags & SHMEMG_AMO_TEST_BEFORE_SWAP) && a.cond == nullptr;
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
    AmoArgs a{w->base, w->stride, sym_off, tgt_pe, elem_idx, (const unsigned long long *)val, val_scalar, nullptr, 0, nullptr, n};
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
              (unsigned long long *)fetched_out, n};
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
              (const unsigned long long *)cond, cond_scalar, (unsigned long long *)fetched_out, n};
    return launch_amo<AMO_CAS>(w, a, idx_bytes, flags, (cudaStream_t)stream);
}
