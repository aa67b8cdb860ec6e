// internal.cuh -- shared declarations of the shmemg CUDA path (sm_100a only).
// Not part of the public boundary (include/shmemg.h); shares nothing with oracle/.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include <map>
#include <string>
#include <vector>

#include "../../include/shmemg.h"

#define SHMEMG_CTL_BYTES (64u * 1024u)     // control region carved from the tail of the slab
#define SHMEMG_ARENA_BYTES (4u << 20)      // plan arena behind the control region: workspace of shmemg_enqueue_batch
#define SHMEMG_STRIDE_ALIGN 512u
#define SHMEMG_MIN_ALIGN 256u
#define SHMEMG_THREADS 256                 // threads per CTA of the register-path copy kernels
#define SHMEMG_TMA_TILE 32768u             // bytes per bulk-copy stage
#define SHMEMG_TMA_STAGES 4                // stages per CTA (128 KiB of shared memory, one CTA per SM)
#define SHMEMG_SIG_SLOTS 1024              // completion counters for single put_signal launches
#define SHMEMG_HOT_MAX 512                 // hot words tracked by SHMEMG_AMO_HOT_AGGREGATE

// ---- control region layout (device) -------------------------------------------------------------------
struct CtlRegion {
    unsigned long long barrier_epoch;      // bumped by barrier_all_on_stream
    unsigned long long bar_arrivals;       // in-kernel barrier: arrivals ever (monotonic, never reset; always a multiple of npes between kernels)
    unsigned int pad[12];
    unsigned int sig_counter[SHMEMG_SIG_SLOTS];   // last-arriver counters of single put_signal launches
    unsigned int group_bar[128];           // per-PE arrival counters of multi-block PE agents (monotonic; halo_app.cu)
    unsigned int amo_done;                 // SHMEMG_AMO_THEN_BARRIER: CTAs of the AMO kernel that have finished
    unsigned int pad_sh;
    unsigned long long shard_bar;          // sharded world: arrivals of every shard's gbarrier (monotonic; system-scope atomics)
    unsigned int hot_n;                    // SHMEMG_AMO_HOT_AGGREGATE: number of hot words found by the sampling kernel
    unsigned int hot_done;                 // CTAs of the sampling kernel that have staged their keys
    unsigned int hot_keys[SHMEMG_HOT_MAX]; // their slab word indices
};

// ---- host-side world ------------------------------------------------------------------------------------
struct shmemg_world {
    int npes = 0;
    int device = 0;
    int sm_count = 0;
    size_t heap_bytes = 0;                 // usable bytes per PE
    size_t stride = 0;                     // distance between PE windows
    uint8_t *base = nullptr;               // DEVICE: window of PE 0
    size_t slab_bytes = 0;
    CtlRegion *ctl = nullptr;              // DEVICE
    std::map<uint64_t, size_t> free_list;  // offset -> size, coalesced
    std::map<uint64_t, size_t> live;       // offset -> size of live allocations
    // the CPU space of the two-space model: npes windows in caller-owned pinned HOST memory
    uint8_t *cpu_base = nullptr;
    size_t cpu_heap_bytes = 0, cpu_stride = 0;
    std::map<uint64_t, size_t> cpu_free_list, cpu_live;
    unsigned sig_seq = 0;
    int ctas_per_sm = 4;                   // copy-class persistent grids: ctas_per_sm * sm_count CTAs
    bool dependent_launch = true;          // executor / planner launches are programmatic dependents (shmemg_set_dependent_launch)
    size_t tile_bytes_override = 0;        // SHMEMG_TILE_BYTES (experiments; forces the register copy path)
    // dynamic shared memory opt-in (cudaFuncSetAttribute) done on THIS world's device, per kernel family
    bool smem_attr_coll = false, smem_attr_probe = false, smem_attr_plan = false, smem_attr_hot = false;
    bool smem_attr_bcast = false, smem_attr_ib = false, smem_attr_shard = false;
    bool smem_attr_red[4][7] = {};         // k_sum_reduce_tma<dtype, op>
    bool smem_attr_set = false;            // the batch executor and the single-copy bulk kernel
    int plan_cluster = 0;                  // CTAs of the device planner's cluster (16, or 8 where 16 cannot be scheduled); 0 = not probed yet
    uint8_t *arena = nullptr;              // DEVICE: plan arena (SHMEMG_ARENA_BYTES) behind the control region
    struct Team { int start, stride, size; };
    int teams_world_npes = 0;              // npes of the world while a team view is active (surface2.cu)
    std::vector<Team> teams;               // user teams (shmemg_team_split_strided); handle = SHMEMG_TEAM_USER0 + index
    // PE -> GPU sharding (shard.cu): this world is shard `shard` of `nshards`; peer_base[s] = slab of shard s as mapped HERE
    int nshards = 0, shard = 0;
    uint8_t *peer_base[SHMEMG_MAX_SHARDS] = {};
    void *peer_ipc[SHMEMG_MAX_SHARDS] = {};   // what cudaIpcOpenMemHandle returned (closed in shmemg_finalize)
    unsigned long long shard_epoch = 0;    // gbarriers enqueued so far
    void *scratch = nullptr;               // DEVICE: caller-owned scratch (shmemg_set_scratch), used by SHMEMG_AMO_HOT_AGGREGATE
    size_t scratch_bytes = 0;
    int amo_last_path = 0;                 // which kernels the last add / fetch-add batch call ran (shmemg_amo_last_path)
    std::string last_cuda_error;
};

static inline int shmemg_cuda_fail(shmemg_world *w, cudaError_t e, const char *what) {
    if (w) w->last_cuda_error = std::string(what) + ": " + cudaGetErrorString(e);
    return SHMEMG_ERR_CUDA;
}
#define SHMEMG_CUDA(w, call)                                              \
    do {                                                                  \
        cudaError_t e__ = (call);                                         \
        if (e__ != cudaSuccess) return shmemg_cuda_fail((w), e__, #call); \
    } while (0)

static inline bool shmemg_in_range(const shmemg_world *w, uint64_t off, uint64_t n) {
    return off <= w->heap_bytes && n <= w->heap_bytes - off;
}
static inline bool shmemg_pe_ok(const shmemg_world *w, int pe) { return pe >= 0 && pe < w->npes; }
// PE -> address translation (a3): base + pe*stride + off
static inline uint8_t *shmemg_addr(const shmemg_world *w, int pe, uint64_t off) {
    return w->base + (size_t)pe * w->stride + off;
}

void shmemg_shard_release(shmemg_world *w);       // shard.cu: closes the peer mappings (shmemg_finalize)

// host-side validation of one op descriptor (batch.cu); shared with the device-initiated interpreter (device_path.cu)
int shmemg_validate_op(const shmemg_world *w, const shmemg_op_t &o);

#ifdef __CUDACC__
// ---- memory-model primitives (GPU scope) --------------------------------------------------------------
__device__ __forceinline__ unsigned ld_acquire_u32(const unsigned *p) {
    unsigned v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ unsigned long long ld_acquire_u64(const unsigned long long *p) {
    unsigned long long v;
    asm volatile("ld.acquire.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}
// polling loads: relaxed (no L1 invalidate per probe); the caller issues ONE fence_acquire() after the poll succeeds
__device__ __forceinline__ unsigned ld_relaxed_u32(const unsigned *p) {
    unsigned v;
    asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ unsigned long long ld_relaxed_u64(const unsigned long long *p) {
    unsigned long long v;
    asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void fence_acquire() { asm volatile("fence.acq_rel.gpu;" ::: "memory"); }
__device__ __forceinline__ void red_release_add_u32(unsigned *p, unsigned v) {
    asm volatile("red.release.gpu.global.add.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
__device__ __forceinline__ void red_release_add_u64(unsigned long long *p, unsigned long long v) {
    asm volatile("red.release.gpu.global.add.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}
__device__ __forceinline__ void exch_release_u64(unsigned long long *p, unsigned long long v) {
    asm volatile("{ .reg .b64 t; atom.release.gpu.global.exch.b64 t, [%0], %1; }" ::"l"(p), "l"(v) : "memory");
}
__device__ __forceinline__ bool cmp_u64(int cmp, unsigned long long s, unsigned long long v) {
    switch (cmp) {
    case SHMEMG_CMP_EQ: return s == v;
    case SHMEMG_CMP_NE: return s != v;
    case SHMEMG_CMP_GT: return s > v;
    case SHMEMG_CMP_GE: return s >= v;
    case SHMEMG_CMP_LT: return s < v;
    default: return s <= v;
    }
}
// signal update with release semantics: visible only after everything the caller has observed
__device__ __forceinline__ void signal_update(unsigned long long *sig, unsigned long long v, int sig_op) {
    if (sig_op == SHMEMG_SIGNAL_ADD) red_release_add_u64(sig, v);
    else exch_release_u64(sig, v);
}


// ---- mbarrier + bulk (TMA) copy primitives: cp.async.bulk moves contiguous 16-byte-aligned blocks between global and
// shared memory without touching registers; one thread drives a whole pipeline (SASS: UBLKCP) -----------------------
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t *b, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(b)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_init_fence() {       // make the initialised barriers visible to the async proxy
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t *b) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(b)) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t *b, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(b)), "r"(bytes) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint64_t *b, unsigned parity) {
    unsigned ok;
    asm volatile("{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.u32 %0, 1, 0, p;\n}"
                 : "=r"(ok) : "r"(smem_u32(b)), "r"(parity) : "memory");
    return ok != 0;
}
// non-blocking probe (try_wait may suspend the thread for an implementation-defined time before returning false)
__device__ __forceinline__ bool mbar_test_wait(uint64_t *b, unsigned parity) {
    unsigned ok;
    asm volatile("{\n .reg .pred p;\n mbarrier.test_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.u32 %0, 1, 0, p;\n}"
                 : "=r"(ok) : "r"(smem_u32(b)), "r"(parity) : "memory");
    return ok != 0;
}
__device__ __forceinline__ void mbar_wait(uint64_t *b, unsigned parity) {
    while (!mbar_test_wait(b, parity)) { }
}
__device__ __forceinline__ void bulk_g2s(void *smem_dst, const void *gsrc, unsigned bytes, uint64_t *full) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(smem_dst)), "l"(gsrc), "r"(bytes), "r"(smem_u32(full)) : "memory");
}
__device__ __forceinline__ void bulk_s2g(void *gdst, const void *smem_src, unsigned bytes) {
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;"
                 ::"l"(gdst), "r"(smem_u32(smem_src)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
// all but the N most recent bulk groups of this thread have finished READING shared memory / have COMPLETED
template <int N> __device__ __forceinline__ void bulk_wait_read() { asm volatile("cp.async.bulk.wait_group.read %0;" ::"n"(N) : "memory"); }
template <int N> __device__ __forceinline__ void bulk_wait() { asm volatile("cp.async.bulk.wait_group %0;" ::"n"(N) : "memory"); }
// order this thread's generic-proxy accesses (acquire loads, release stores) against its async-proxy (bulk) accesses
__device__ __forceinline__ void proxy_fence() { asm volatile("fence.proxy.async;" ::: "memory"); }
__device__ __forceinline__ void named_bar_sync(int id, int nthreads) {
    asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}

// ---- streaming 128-bit accesses: L2-coherent loads (never a stale L1 line), evict-first hints --------------
__device__ __forceinline__ int4 ld_stream16(const void *p) {
    int4 r;
    asm volatile("ld.global.cg.v4.s32 {%0,%1,%2,%3}, [%4];" : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p));
    return r;
}
__device__ __forceinline__ void st_stream16(void *p, const int4 &v) {
    asm volatile("st.global.cg.v4.s32 [%0], {%1,%2,%3,%4};" ::"l"(p), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
}

template <typename T>
__device__ __forceinline__ void copy_elems(uint8_t *dst, const uint8_t *src, size_t n, int tid, int nthr) {
    T *d = reinterpret_cast<T *>(dst);
    const volatile T *s = reinterpret_cast<const volatile T *>(src);
    for (size_t i = tid; i < n; i += nthr) d[i] = s[i];
}

// Cooperative copy of n bytes, any alignment, by threads tid in [0, nthr).  Fast path: dst and src are
// congruent mod 16 -> byte head, unrolled 128-bit body, byte tail.  Otherwise the widest element the
// relative misalignment allows.  All loads bypass L1 (coherent at L2).
template <int UNROLL>
__device__ __forceinline__ void copy_coop(uint8_t *dst, const uint8_t *src, size_t n, int tid, int nthr) {
    if (n == 0) return;
    const unsigned rel = (unsigned)((reinterpret_cast<uintptr_t>(dst) ^ reinterpret_cast<uintptr_t>(src)) & 15u);
    if (rel == 0) {
        size_t head = (16u - (unsigned)(reinterpret_cast<uintptr_t>(dst) & 15u)) & 15u;
        if (head > n) head = n;
        if (tid < (int)head) dst[tid] = *reinterpret_cast<const volatile uint8_t *>(src + tid);
        const size_t nvec = (n - head) >> 4;
        int4 *d = reinterpret_cast<int4 *>(dst + head);
        const int4 *s = reinterpret_cast<const int4 *>(src + head);
        size_t i = tid;
        const size_t step = (size_t)UNROLL * nthr;
        for (; i + (size_t)(UNROLL - 1) * nthr < nvec; i += step) {
            int4 v[UNROLL];
#pragma unroll
            for (int u = 0; u < UNROLL; ++u) v[u] = ld_stream16(s + i + (size_t)u * nthr);
#pragma unroll
            for (int u = 0; u < UNROLL; ++u) st_stream16(d + i + (size_t)u * nthr, v[u]);
        }
        for (; i < nvec; i += nthr) st_stream16(d + i, ld_stream16(s + i));
        const size_t done = head + (nvec << 4);
        const size_t tail = n - done;
        if (tid < (int)tail) dst[done + tid] = *reinterpret_cast<const volatile uint8_t *>(src + done + tid);
        return;
    }
    // relative misalignment: align dst to W, copy W-byte elements, byte head/tail
    const unsigned W = (rel & 7u) == 0 ? 8u : (rel & 3u) == 0 ? 4u : (rel & 1u) == 0 ? 2u : 1u;
    size_t head = (W - (unsigned)(reinterpret_cast<uintptr_t>(dst) & (W - 1u))) & (W - 1u);
    if (head > n) head = n;
    if (tid < (int)head) dst[tid] = *reinterpret_cast<const volatile uint8_t *>(src + tid);
    const size_t nel = (n - head) / W;
    switch (W) {
    case 8: copy_elems<unsigned long long>(dst + head, src + head, nel, tid, nthr); break;
    case 4: copy_elems<unsigned int>(dst + head, src + head, nel, tid, nthr); break;
    case 2: copy_elems<unsigned short>(dst + head, src + head, nel, tid, nthr); break;
    default: copy_elems<unsigned char>(dst + head, src + head, nel, tid, nthr); break;
    }
    const size_t done = head + nel * W;
    const size_t tail = n - done;
    if (tid < (int)tail) dst[done + tid] = *reinterpret_cast<const volatile uint8_t *>(src + done + tid);
}
#endif  // __CUDACC__
