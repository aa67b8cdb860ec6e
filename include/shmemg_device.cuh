/*
 * shmemg_device.cuh -- DEVICE-INITIATED entry points (Tier-1) of the B200-native GPU-aware OpenSHMEM hot path.
 *
 * Header-only `__device__` functions for CUDA kernels compiled for sm_100a.  They are the device-side counterparts
 * of the `_on_stream` routines of shmemg.h: "device-initiated communication [is] invoked from GPU kernels"
 * (PAPER L142, L271, L465-L466), uses the default device context (`SHMEM_DEVICE_CTX_DEFAULT`: "device
 * code that omits an explicit context uses" it) and the world team (`SHMEM_DEVICE_TEAM_WORLD`, L194, L357).
 *
 * Model
 *   - The kernel receives a `shmemg_device_world_t` BY VALUE (filled on the host by shmemg_device_world_get); it holds
 *     the slab base, the window stride and the npes of the world: PE -> address translation is
 *     base + pe*stride + off, two integer operations and no pointer classification in device code (L351).
 *   - All N PEs share the GPU, so every routine takes the initiating PE `pe` explicitly, like the host API.
 *     Operands are symmetric offsets (L287, L355); AMO values are immediates.
 *   - THREAD COLLABORATION: a routine without suffix is called by ONE thread and acts
 *     for it alone; `_warp` / `_block` routines must be called by ALL threads of the warp / thread block with the
 *     same arguments ("uniform participation"), they share the work and return to all of them.  Mixing scopes on
 *     one operation, or divergent participation, is undefined (L371).
 *   - COMPLETION (L367-L369): put/get return on LOCAL completion (the source may be reused; a get's data may be
 *     read by the calling thread / after the routine's closing barrier by the calling group).  Remote visibility and
 *     ordering need shmemg_dev_fence / shmemg_dev_quiet (L377: "GPU implementations may use weaker default ordering,
 *     provided fence and quiet restore ordering").  "Atomicity does not imply ordering" (L365).
 *   - put_signal: the signal word update is atomic w.r.t. other signal updates and waits and becomes visible only
 *     after the whole payload (release at GPU scope; L218, L461).  signal_wait_until polls with acquire semantics.
 *   - barrier_all_block is a DEVICE COLLECTIVE: it needs one participating thread block per PE, all co-resident
 *     (cooperative launch) -- progress of a spinning kernel is otherwise not guaranteed (L214, L394, L477).
 *   - Host visibility of device-initiated updates still needs host-side synchronisation of the stream (L388-L390).
 *   - Errors: none are reported on the device; out-of-range PEs/offsets and misaligned AMO words are undefined
 *     behaviour (L435).
 */
#ifndef SHMEMG_DEVICE_CUH
#define SHMEMG_DEVICE_CUH

#include "shmemg.h"

#if defined(__CUDACC__)

/* ---- address translation (shmem_ptr analog on the device) ------------------------------------ */
__device__ __forceinline__ unsigned char *shmemg_dev_ptr(const shmemg_device_world_t &w, uint64_t sym_off, int pe) {
    return w.base + (size_t)pe * w.stride + sym_off;
}
__device__ __forceinline__ int shmemg_dev_n_pes(const shmemg_device_world_t &w) { return w.npes; }

/* ---- memory-model primitives (GPU scope) ------------------------------------------------------------------------ */
__device__ __forceinline__ void shmemg_dev_fence_gpu() { asm volatile("fence.acq_rel.gpu;" ::: "memory"); }
__device__ __forceinline__ unsigned long long shmemg_dev_ld_relaxed(const unsigned long long *p) {
    unsigned long long v;
    asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ bool shmemg_dev_cmp(int cmp, unsigned long long s, unsigned long long v) {
    switch (cmp) {
    case SHMEMG_CMP_EQ: return s == v;
    case SHMEMG_CMP_NE: return s != v;
    case SHMEMG_CMP_GT: return s > v;
    case SHMEMG_CMP_GE: return s >= v;
    case SHMEMG_CMP_LT: return s < v;
    default: return s <= v;
    }
}

/* ---- cooperative copy: threads tid in [0, nthr) move n bytes, any alignment ------------------------------------
 * Every naturally aligned 1/2/4/8/16-byte unit that both addresses allow is moved by ONE access of that width, so an
 * aligned 8-byte put used as a flag is never torn.  Loads bypass L1 (coherent at L2). */
template <typename T>
__device__ __forceinline__ void shmemg_dev_copy_elems(unsigned char *d, const unsigned char *s, size_t nel, int tid, int nthr) {
    T *dd = reinterpret_cast<T *>(d);
    const volatile T *ss = reinterpret_cast<const volatile T *>(s);
    for (size_t i = tid; i < nel; i += nthr) dd[i] = ss[i];
}
__device__ __forceinline__ void shmemg_dev_copy_w(unsigned char *d, const unsigned char *s, size_t n, unsigned W, int tid, int nthr) {
    switch (W) {
    case 8: shmemg_dev_copy_elems<unsigned long long>(d, s, n >> 3, tid, nthr); break;
    case 4: shmemg_dev_copy_elems<unsigned int>(d, s, n >> 2, tid, nthr); break;
    case 2: shmemg_dev_copy_elems<unsigned short>(d, s, n >> 1, tid, nthr); break;
    default: shmemg_dev_copy_elems<unsigned char>(d, s, n, tid, nthr); break;
    }
}
__device__ __forceinline__ void shmemg_dev_copy(unsigned char *dst, const unsigned char *src, size_t n, int tid, int nthr) {
    if (n == 0) return;
    const uintptr_t da = reinterpret_cast<uintptr_t>(dst), sa = reinterpret_cast<uintptr_t>(src);
    const unsigned both = (unsigned)((da | sa) & 15u);
    /* W = widest power of two (<= 16) dividing both addresses */
    unsigned W = both == 0 ? 16u : (both & (0u - both));
    if (W < 16u && ((da ^ sa) & 15u) == 0 && n >= 32) {
        /* congruent mod 16: a short W-wide head reaches 16-byte alignment, then the vector body below */
        const size_t head = (16u - (unsigned)(da & 15u)) & 15u;
        shmemg_dev_copy_w(dst, src, head, W, tid, nthr);
        dst += head; src += head; n -= head;
        W = 16u;
    }
    size_t body;
    if (W == 16u) {
        body = n & ~(size_t)15;
        int4 *d4 = reinterpret_cast<int4 *>(dst);
        const int4 *s4 = reinterpret_cast<const int4 *>(src);
        for (size_t i = tid; i < (body >> 4); i += nthr) {
            int4 v;
            asm volatile("ld.global.cg.v4.s32 {%0,%1,%2,%3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(s4 + i));
            d4[i] = v;
        }
    } else {
        body = n & ~(size_t)(W - 1u);
        shmemg_dev_copy_w(dst, src, body, W, tid, nthr);
    }
    /* tail < W bytes: aligned to W at its start, so 8/4/2/1-byte units in descending order stay naturally aligned */
    size_t off = body, left = n - body;
    for (unsigned u = 8; u >= 1; u >>= 1) {
        if (u < W && left >= u) {
            if (tid == 0) shmemg_dev_copy_w(dst + off, src + off, u, u, 0, 1);
            off += u; left -= u;
        }
    }
}

/* ---- put / get: thread, warp and block scope ---------------------------------------------------------
 * put: heap[target_pe][dest_off ..] = heap[pe][source_off ..];  get: heap[pe][dest_off ..] = heap[target_pe][source_off ..] */
__device__ __forceinline__ void shmemg_dev_put(const shmemg_device_world_t &w, uint64_t dest_off, uint64_t source_off,
                                               size_t nbytes, int pe, int target_pe) {
    shmemg_dev_copy(shmemg_dev_ptr(w, dest_off, target_pe), shmemg_dev_ptr(w, source_off, pe), nbytes, 0, 1);
}
__device__ __forceinline__ void shmemg_dev_get(const shmemg_device_world_t &w, uint64_t dest_off, uint64_t source_off,
                                               size_t nbytes, int pe, int target_pe) {
    shmemg_dev_copy(shmemg_dev_ptr(w, dest_off, pe), shmemg_dev_ptr(w, source_off, target_pe), nbytes, 0, 1);
}
__device__ __forceinline__ void shmemg_dev_put_warp(const shmemg_device_world_t &w, uint64_t dest_off, uint64_t source_off,
                                                    size_t nbytes, int pe, int target_pe) {
    shmemg_dev_copy(shmemg_dev_ptr(w, dest_off, target_pe), shmemg_dev_ptr(w, source_off, pe), nbytes, threadIdx.x & 31, 32);
    __syncwarp();
}
__device__ __forceinline__ void shmemg_dev_get_warp(const shmemg_device_world_t &w, uint64_t dest_off, uint64_t source_off,
                                                    size_t nbytes, int pe, int target_pe) {
    shmemg_dev_copy(shmemg_dev_ptr(w, dest_off, pe), shmemg_dev_ptr(w, source_off, target_pe), nbytes, threadIdx.x & 31, 32);
    __syncwarp();
}
__device__ __forceinline__ int shmemg_dev_block_tid() {
    return (int)(threadIdx.x + blockDim.x * (threadIdx.y + blockDim.y * threadIdx.z));
}
__device__ __forceinline__ int shmemg_dev_block_size() { return (int)(blockDim.x * blockDim.y * blockDim.z); }
__device__ __forceinline__ void shmemg_dev_put_block(const shmemg_device_world_t &w, uint64_t dest_off, uint64_t source_off,
                                                     size_t nbytes, int pe, int target_pe) {
    shmemg_dev_copy(shmemg_dev_ptr(w, dest_off, target_pe), shmemg_dev_ptr(w, source_off, pe), nbytes,
                    shmemg_dev_block_tid(), shmemg_dev_block_size());
    __syncthreads();
}
__device__ __forceinline__ void shmemg_dev_get_block(const shmemg_device_world_t &w, uint64_t dest_off, uint64_t source_off,
                                                     size_t nbytes, int pe, int target_pe) {
    shmemg_dev_copy(shmemg_dev_ptr(w, dest_off, pe), shmemg_dev_ptr(w, source_off, target_pe), nbytes,
                    shmemg_dev_block_tid(), shmemg_dev_block_size());
    __syncthreads();
}

/* ---- ordering: fence orders, quiet completes; here both are one GPU-scope fence ------------------
 * Stores and atomics issued by the calling thread before the call are visible at GPU scope before anything it
 * issues afterwards (the strong reading of L377: all targets, gets and atomics included).  The `_block` forms are
 * for the block-scope put/get above: every thread of the block fences its own share, then the block synchronises, so
 * that whatever ANY thread of the block issues afterwards is ordered after the whole block's earlier operations. */
__device__ __forceinline__ void shmemg_dev_fence() { shmemg_dev_fence_gpu(); }
__device__ __forceinline__ void shmemg_dev_quiet() { shmemg_dev_fence_gpu(); }
__device__ __forceinline__ void shmemg_dev_fence_warp() { shmemg_dev_fence_gpu(); __syncwarp(); }
__device__ __forceinline__ void shmemg_dev_quiet_warp() { shmemg_dev_fence_gpu(); __syncwarp(); }
__device__ __forceinline__ void shmemg_dev_fence_block() { shmemg_dev_fence_gpu(); __syncthreads(); }
__device__ __forceinline__ void shmemg_dev_quiet_block() { shmemg_dev_fence_gpu(); __syncthreads(); }

/* ---- signals ----------------------------------------------------------------------------- */
__device__ __forceinline__ void shmemg_dev_signal_update(unsigned long long *sig, uint64_t value, int sig_op) {
    if (sig_op == SHMEMG_SIGNAL_ADD)
        asm volatile("red.release.gpu.global.add.u64 [%0], %1;" ::"l"(sig), "l"(value) : "memory");
    else
        asm volatile("{ .reg .b64 t; atom.release.gpu.global.exch.b64 t, [%0], %1; }" ::"l"(sig), "l"(value) : "memory");
}
/* thread scope: payload by the calling thread, then the signal with release semantics */
__device__ __forceinline__ void shmemg_dev_put_signal(const shmemg_device_world_t &w, uint64_t dest_off, uint64_t source_off,
                                                      size_t nbytes, uint64_t sig_off, uint64_t signal, int sig_op, int pe,
                                                      int target_pe) {
    shmemg_dev_put(w, dest_off, source_off, nbytes, pe, target_pe);
    shmemg_dev_signal_update(reinterpret_cast<unsigned long long *>(shmemg_dev_ptr(w, sig_off, target_pe)), signal, sig_op);
}
/* block scope: all threads copy, every thread fences its share, the block synchronises, one thread signals */
__device__ __forceinline__ void shmemg_dev_put_signal_block(const shmemg_device_world_t &w, uint64_t dest_off,
                                                            uint64_t source_off, size_t nbytes, uint64_t sig_off,
                                                            uint64_t signal, int sig_op, int pe, int target_pe) {
    shmemg_dev_copy(shmemg_dev_ptr(w, dest_off, target_pe), shmemg_dev_ptr(w, source_off, pe), nbytes,
                    shmemg_dev_block_tid(), shmemg_dev_block_size());
    shmemg_dev_fence_gpu();
    __syncthreads();
    if (shmemg_dev_block_tid() == 0)
        shmemg_dev_signal_update(reinterpret_cast<unsigned long long *>(shmemg_dev_ptr(w, sig_off, target_pe)), signal, sig_op);
}
/* block scope, block-strided (ibput analog): for b < nblocks: dest[b*dst_stride .. +block_bytes) on `target_pe` =
 * source[b*src_stride .. +block_bytes) on `pe`; strides in bytes.  8-byte aligned blocks move one 64-bit word per thread
 * (the contiguous side coalesces), anything else goes block by block through the any-alignment copy. */
__device__ __forceinline__ void shmemg_dev_ibput_block(const shmemg_device_world_t &w, uint64_t dest_off, uint64_t source_off,
                                                       uint64_t dst_stride, uint64_t src_stride, size_t block_bytes,
                                                       size_t nblocks, int pe, int target_pe) {
    unsigned char *d = shmemg_dev_ptr(w, dest_off, target_pe);
    const unsigned char *s = shmemg_dev_ptr(w, source_off, pe);
    const int tid = shmemg_dev_block_tid(), nthr = shmemg_dev_block_size();
    if (((reinterpret_cast<uintptr_t>(d) | reinterpret_cast<uintptr_t>(s) | dst_stride | src_stride | block_bytes) & 7) == 0) {
        const size_t wpb = block_bytes >> 3, nw = nblocks * wpb;
#pragma unroll 1
        for (size_t e0 = tid; e0 < nw; e0 += (size_t)4 * nthr) {          /* four independent words in flight per thread */
            unsigned long long v[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const size_t e = e0 + (size_t)u * nthr, b = e / wpb, k = e - b * wpb;
                if (e < nw) v[u] = *reinterpret_cast<const volatile unsigned long long *>(s + b * src_stride + 8 * k);
            }
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const size_t e = e0 + (size_t)u * nthr, b = e / wpb, k = e - b * wpb;
                if (e < nw) *reinterpret_cast<unsigned long long *>(d + b * dst_stride + 8 * k) = v[u];
            }
        }
    } else {
        for (size_t b = 0; b < nblocks; ++b) shmemg_dev_copy(d + b * dst_stride, s + b * src_stride, block_bytes, tid, nthr);
    }
    __syncthreads();
}
/* block scope: signal only -- everything the BLOCK has put before becomes visible on target_pe before the signal */
__device__ __forceinline__ void shmemg_dev_signal_block(const shmemg_device_world_t &w, uint64_t sig_off, uint64_t signal,
                                                        int sig_op, int target_pe) {
    shmemg_dev_fence_gpu();
    __syncthreads();
    if (shmemg_dev_block_tid() == 0)
        shmemg_dev_signal_update(reinterpret_cast<unsigned long long *>(shmemg_dev_ptr(w, sig_off, target_pe)), signal, sig_op);
}
/* blocks the calling thread until cmp(u64 heap[pe][sig_off], value) holds (unsigned compare); what it reads afterwards
 * is at least as new as what the signalling put_signal released */
__device__ __forceinline__ uint64_t shmemg_dev_signal_wait_until(const shmemg_device_world_t &w, uint64_t sig_off, int cmp,
                                                                 uint64_t value, int pe) {
    const unsigned long long *sig = reinterpret_cast<const unsigned long long *>(shmemg_dev_ptr(w, sig_off, pe));
    unsigned long long s;
    while (!shmemg_dev_cmp(cmp, s = shmemg_dev_ld_relaxed(sig), value)) __nanosleep(32);
    shmemg_dev_fence_gpu();
    return s;
}
/* non-blocking probe of the same condition (shmem_signal_test analog): 1 if it holds (then acquire), else 0 */
__device__ __forceinline__ int shmemg_dev_signal_test(const shmemg_device_world_t &w, uint64_t sig_off, int cmp, uint64_t value,
                                                      int pe) {
    const unsigned long long *sig = reinterpret_cast<const unsigned long long *>(shmemg_dev_ptr(w, sig_off, pe));
    if (!shmemg_dev_cmp(cmp, shmemg_dev_ld_relaxed(sig), value)) return 0;
    shmemg_dev_fence_gpu();
    return 1;
}
/* block scope: one thread polls, the block synchronises; every thread may read the payload afterwards */
__device__ __forceinline__ void shmemg_dev_signal_wait_until_block(const shmemg_device_world_t &w, uint64_t sig_off, int cmp,
                                                                   uint64_t value, int pe) {
    if (shmemg_dev_block_tid() == 0) shmemg_dev_signal_wait_until(w, sig_off, cmp, value, pe);
    __syncthreads();
}

/* ---- atomics on 64-bit words, thread scope, relaxed: atomicity does not imply ordering -------
 * add: red.global (nothing fetched); fetch_add / compare_swap: atom.global (old value returned). */
__device__ __forceinline__ void shmemg_dev_atomic_add(const shmemg_device_world_t &w, uint64_t dest_off, uint64_t value,
                                                      int target_pe) {
    asm volatile("red.relaxed.gpu.global.add.u64 [%0], %1;" ::"l"(shmemg_dev_ptr(w, dest_off, target_pe)), "l"(value) : "memory");
}
__device__ __forceinline__ uint64_t shmemg_dev_atomic_fetch_add(const shmemg_device_world_t &w, uint64_t dest_off,
                                                                uint64_t value, int target_pe) {
    unsigned long long old;
    asm volatile("atom.relaxed.gpu.global.add.u64 %0, [%1], %2;" : "=l"(old)
                 : "l"(shmemg_dev_ptr(w, dest_off, target_pe)), "l"(value) : "memory");
    return old;
}
__device__ __forceinline__ uint64_t shmemg_dev_atomic_compare_swap(const shmemg_device_world_t &w, uint64_t dest_off,
                                                                   uint64_t cond, uint64_t value, int target_pe) {
    unsigned long long old;
    asm volatile("atom.relaxed.gpu.global.cas.b64 %0, [%1], %2, %3;" : "=l"(old)
                 : "l"(shmemg_dev_ptr(w, dest_off, target_pe)), "l"(cond), "l"(value) : "memory");
    return old;
}

/* ---- device barrier (device collective, Table 6 "uniform participation") ---------------------------
 * Called by ALL threads of ONE thread block per PE; the npes blocks must be co-resident (cooperative launch).
 * Implies quiet for every PE: all updates issued before the barrier by any participating block are visible to all
 * of them after it.  ONE monotonic arrival counter in the world's control region (never reset, 64 bits): an agent arrives with a
 * fire-and-forget release `red` and polls the counter itself until it has reached the end of the current round of npes
 * arrivals -- no atomic return value to wait for, no last arriver, no second word (1.17 us per barrier for 128 agents against
 * 1.83 us for a sense-reversing counter + generation word).  The round is found from the counter alone: before its own arrival
 * to barrier k an agent can only read a value in [k*npes, (k+1)*npes), whatever the others have done.  Do not run it
 * concurrently with shmemg_barrier_all_repeat_on_stream or a second device kernel of the same world. */
__device__ __forceinline__ void shmemg_dev_barrier_all_block(const shmemg_device_world_t &w) {
    shmemg_dev_fence_gpu();                 /* every thread: its own earlier updates */
    __syncthreads();
    if (shmemg_dev_block_tid() == 0) {
        /* the load is issued first and consumed only by the poll: the arrival does not wait for it */
        unsigned long long cnt;
        asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(cnt) : "l"(w.bar_arrivals) : "memory");
        asm volatile("red.release.gpu.global.add.u64 [%0], %1;" ::"l"(w.bar_arrivals), "l"(1ull) : "memory");
        const unsigned long long target = cnt - cnt % (unsigned long long)w.npes + (unsigned long long)w.npes;
        unsigned long long c;
        do {
            asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(c) : "l"(w.bar_arrivals) : "memory");
        } while (c < target);
        shmemg_dev_fence_gpu();
    }
    __syncthreads();
}

/* ---- explicit contexts and non-blocking operations (see shmemg.h "explicit device contexts") -------
 * A context's queue holds the PE's pending non-blocking operations; `counters[0]` counts the operations issued on it,
 * `counters[1]` those completed.  Thread scope: ONE thread uses the context; `_block`: all threads of the block, same arguments. */
__device__ __forceinline__ unsigned long long shmemg_dev_ctx_issued(const shmemg_device_ctx_t &c) {
    return *reinterpret_cast<volatile unsigned long long *>(c.counters);
}
__device__ __forceinline__ unsigned long long shmemg_dev_ctx_completed(const shmemg_device_ctx_t &c) {
    return *reinterpret_cast<volatile unsigned long long *>(c.counters + 1);
}
__device__ __forceinline__ unsigned long long shmemg_dev_ctx_pending(const shmemg_device_ctx_t &c) {
    return shmemg_dev_ctx_issued(c) - shmemg_dev_ctx_completed(c);
}
/* perform the pending operations of the context in issue order (threads tid of nthr cooperate); then one GPU-scope fence */
__device__ __forceinline__ void shmemg_dev_ctx_drain(const shmemg_device_ctx_t &c, int tid, int nthr) {
    const unsigned long long issued = shmemg_dev_ctx_issued(c), done = shmemg_dev_ctx_completed(c);
    for (unsigned long long k = done; k < issued; ++k) {
        const shmemg_nbi_rec_t r = c.queue[k % c.capacity];
        shmemg_dev_copy(reinterpret_cast<unsigned char *>(r.dst), reinterpret_cast<const unsigned char *>(r.src), (size_t)r.nbytes, tid, nthr);
        if (r.sig) {                                  /* put_signal: the signal after the whole payload */
            shmemg_dev_fence_gpu();
            if (nthr > 1) __syncthreads();
            if (tid == 0) shmemg_dev_signal_update(reinterpret_cast<unsigned long long *>(r.sig), r.sig_value, (int)r.sig_op);
        }
    }
    shmemg_dev_fence_gpu();
}
/* quiet: every operation issued on THIS context is complete and visible; other contexts of the PE are left alone */
__device__ __forceinline__ void shmemg_dev_ctx_quiet(const shmemg_device_ctx_t &c) {
    shmemg_dev_ctx_drain(c, 0, 1);
    *reinterpret_cast<volatile unsigned long long *>(c.counters + 1) = shmemg_dev_ctx_issued(c);
}
__device__ __forceinline__ void shmemg_dev_ctx_quiet_block(const shmemg_device_ctx_t &c) {
    __syncthreads();
    shmemg_dev_ctx_drain(c, shmemg_dev_block_tid(), shmemg_dev_block_size());
    __syncthreads();
    if (shmemg_dev_block_tid() == 0) *reinterpret_cast<volatile unsigned long long *>(c.counters + 1) = shmemg_dev_ctx_issued(c);
    __syncthreads();
}
/* fence: operations issued on this context afterwards are delivered after the earlier ones.  The pending ones are delivered
 * here (always conformant: stronger than required) */
__device__ __forceinline__ void shmemg_dev_ctx_fence(const shmemg_device_ctx_t &c) { shmemg_dev_ctx_quiet(c); }
__device__ __forceinline__ void shmemg_dev_ctx_fence_block(const shmemg_device_ctx_t &c) { shmemg_dev_ctx_quiet_block(c); }
/* record one operation; a full queue is drained first (a non-blocking operation may complete at any time before the quiet) */
__device__ __forceinline__ void shmemg_dev_ctx_push(const shmemg_device_ctx_t &c, const shmemg_nbi_rec_t &r) {
    if (shmemg_dev_ctx_pending(c) >= c.capacity) shmemg_dev_ctx_quiet(c);
    const unsigned long long k = shmemg_dev_ctx_issued(c);
    c.queue[k % c.capacity] = r;
    *reinterpret_cast<volatile unsigned long long *>(c.counters) = k + 1;
}
__device__ __forceinline__ void shmemg_dev_put_nbi(const shmemg_device_world_t &w, const shmemg_device_ctx_t &c, uint64_t dest_off,
                                                   uint64_t source_off, size_t nbytes, int target_pe) {
    shmemg_nbi_rec_t r = {};
    r.dst = (uint64_t)shmemg_dev_ptr(w, dest_off, target_pe); r.src = (uint64_t)shmemg_dev_ptr(w, source_off, c.pe); r.nbytes = nbytes;
    shmemg_dev_ctx_push(c, r);
}
__device__ __forceinline__ void shmemg_dev_get_nbi(const shmemg_device_world_t &w, const shmemg_device_ctx_t &c, uint64_t dest_off,
                                                   uint64_t source_off, size_t nbytes, int target_pe) {
    shmemg_nbi_rec_t r = {};
    r.dst = (uint64_t)shmemg_dev_ptr(w, dest_off, c.pe); r.src = (uint64_t)shmemg_dev_ptr(w, source_off, target_pe); r.nbytes = nbytes;
    shmemg_dev_ctx_push(c, r);
}
__device__ __forceinline__ void shmemg_dev_put_signal_nbi(const shmemg_device_world_t &w, const shmemg_device_ctx_t &c, uint64_t dest_off,
                                                          uint64_t source_off, size_t nbytes, uint64_t sig_off, uint64_t signal,
                                                          int sig_op, int target_pe) {
    shmemg_nbi_rec_t r = {};
    r.dst = (uint64_t)shmemg_dev_ptr(w, dest_off, target_pe); r.src = (uint64_t)shmemg_dev_ptr(w, source_off, c.pe); r.nbytes = nbytes;
    r.sig = (uint64_t)shmemg_dev_ptr(w, sig_off, target_pe); r.sig_value = signal; r.sig_op = (uint32_t)sig_op;
    shmemg_dev_ctx_push(c, r);
}

/* ---- device collectives (PAPER L226 case study 3 "thread-collaborative collective reductions", L363-L371, Table 6 "Device
 * collectives: if provided, uniform participation") ------------------------------------------------------------------------
 * Block scope, ONE thread block per PE: ALL npes blocks (co-resident: cooperative launch) call the routine with the same
 * arguments except `pe`, every thread of each block takes part.  Each routine is a barrier on entry (every PE's source is
 * complete) and on exit (every PE's dest is complete and visible to every PE).  Same definitions as the stream collectives of
 * shmemg.h; source and dest ranges must not overlap (sum_reduce: dest == source allowed). */

/* every PE's dest[k] = sum over PEs (ascending) of source[k].  Reduce-scatter + all-gather: block p sums the p-th share of the
 * elements over all N windows (fp32: fp64 accumulation, one rounding -- bit-equal to the stream collective) and stores the result
 * into all N windows, so every element is read N times and written N times in total, the same traffic as k_sum_reduce_tma. */
template <typename T, typename ACC>
__device__ __forceinline__ void shmemg_dev_sum_share(const shmemg_device_world_t &w, uint64_t dest_off, uint64_t source_off,
                                                     size_t lo, size_t hi, int tid, int nthr) {
    for (size_t k = lo + tid; k < hi; k += nthr) {
        ACC acc = (ACC)0;
        for (int q = 0; q < w.npes; ++q)
            acc += (ACC) * reinterpret_cast<const volatile T *>(shmemg_dev_ptr(w, source_off, q) + k * sizeof(T));
        const T r = (T)acc;
        for (int j = 0; j < w.npes; ++j) *reinterpret_cast<T *>(shmemg_dev_ptr(w, dest_off, j) + k * sizeof(T)) = r;
    }
}
__device__ __forceinline__ void shmemg_dev_sum_reduce_block(const shmemg_device_world_t &w, int dtype, uint64_t dest_off,
                                                            uint64_t source_off, size_t nreduce, int pe) {
    shmemg_dev_barrier_all_block(w);
    const int tid = shmemg_dev_block_tid(), nthr = shmemg_dev_block_size();
    const size_t per = (nreduce + (size_t)w.npes - 1) / (size_t)w.npes;
    const size_t lo = per * (size_t)pe < nreduce ? per * (size_t)pe : nreduce, hi = lo + per < nreduce ? lo + per : nreduce;
    if (dtype == SHMEMG_F32) {
        /* four columns per thread and PE: 16-byte loads when the share is aligned, ascending PE order, fp64 accumulators */
        const bool vec = ((dest_off | source_off | (uint64_t)w.stride | (uint64_t)(uintptr_t)w.base) & 15) == 0 && (lo & 3) == 0;
        size_t done = lo;
        if (vec) {
            const size_t nv = (hi - lo) >> 2;
            for (size_t v = tid; v < nv; v += nthr) {
                double a0 = 0.0, a1 = 0.0, a2 = 0.0, a3 = 0.0;
                const size_t byte = (lo + 4 * v) * 4;
#pragma unroll 4
                for (int q = 0; q < w.npes; ++q) {
                    float4 x;
                    asm volatile("ld.global.cg.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(x.x), "=f"(x.y), "=f"(x.z), "=f"(x.w)
                                 : "l"(shmemg_dev_ptr(w, source_off, q) + byte));
                    a0 += (double)x.x; a1 += (double)x.y; a2 += (double)x.z; a3 += (double)x.w;
                }
                const float4 r = make_float4((float)a0, (float)a1, (float)a2, (float)a3);
                for (int j = 0; j < w.npes; ++j) *reinterpret_cast<float4 *>(shmemg_dev_ptr(w, dest_off, j) + byte) = r;
            }
            done = lo + (nv << 2);
        }
        shmemg_dev_sum_share<float, double>(w, dest_off, source_off, done, hi, tid, nthr);
    } else if (dtype == SHMEMG_I64) {
        shmemg_dev_sum_share<unsigned long long, unsigned long long>(w, dest_off, source_off, lo, hi, tid, nthr);
    } else if (dtype == SHMEMG_I32) {
        shmemg_dev_sum_share<unsigned, unsigned>(w, dest_off, source_off, lo, hi, tid, nthr);
    } else {
        shmemg_dev_sum_share<double, double>(w, dest_off, source_off, lo, hi, tid, nthr);
    }
    shmemg_dev_barrier_all_block(w);
}
/* every PE's dest[p*nbytes .. +nbytes) = PE p's source: block p puts its block into all N windows */
__device__ __forceinline__ void shmemg_dev_fcollect_block(const shmemg_device_world_t &w, uint64_t dest_off, uint64_t source_off,
                                                          size_t nbytes, int pe) {
    shmemg_dev_barrier_all_block(w);
    const int tid = shmemg_dev_block_tid(), nthr = shmemg_dev_block_size();
    for (int j = 0; j < w.npes; ++j)
        shmemg_dev_copy(shmemg_dev_ptr(w, dest_off + (uint64_t)pe * nbytes, j), shmemg_dev_ptr(w, source_off, pe), nbytes, tid, nthr);
    shmemg_dev_barrier_all_block(w);
}
/* PE j's dest[i*nbytes .. +nbytes) = PE i's source[j*nbytes .. +nbytes): block i puts its N blocks */
__device__ __forceinline__ void shmemg_dev_alltoall_block(const shmemg_device_world_t &w, uint64_t dest_off, uint64_t source_off,
                                                          size_t nbytes, int pe) {
    shmemg_dev_barrier_all_block(w);
    const int tid = shmemg_dev_block_tid(), nthr = shmemg_dev_block_size();
    for (int j = 0; j < w.npes; ++j)
        shmemg_dev_copy(shmemg_dev_ptr(w, dest_off + (uint64_t)pe * nbytes, j), shmemg_dev_ptr(w, source_off + (uint64_t)j * nbytes, pe),
                        nbytes, tid, nthr);
    shmemg_dev_barrier_all_block(w);
}
/* every PE's dest = the root's source: every block gets the root's block (the root's own dest included) */
__device__ __forceinline__ void shmemg_dev_broadcast_block(const shmemg_device_world_t &w, uint64_t dest_off, uint64_t source_off,
                                                           size_t nbytes, int root_pe, int pe) {
    shmemg_dev_barrier_all_block(w);
    shmemg_dev_copy(shmemg_dev_ptr(w, dest_off, pe), shmemg_dev_ptr(w, source_off, root_pe), nbytes, shmemg_dev_block_tid(),
                    shmemg_dev_block_size());
    shmemg_dev_barrier_all_block(w);
}

#endif /* __CUDACC__ */
#endif /* SHMEMG_DEVICE_CUH */
