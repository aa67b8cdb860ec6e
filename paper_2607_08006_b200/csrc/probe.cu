// probe.cu -- ceiling probes (include/shmemg_probe.h): bare L2 atomics at hashed addresses and a plain
// per-PE local copy.  Measurement utilities for bench.py; not operations of the specification.
#include "tma_stream.cuh"
#include "../../include/shmemg_probe.h"

__device__ __forceinline__ unsigned long long probe_hash(unsigned long long i) {
    unsigned long long x = i * 0x9E3779B97F4A7C15ull + 0x632BE59BD9B4E019ull;
    x ^= x >> 29; x *= 0xBF58476D1CE4E5B9ull;
    x ^= x >> 32;
    return x;
}

template <int MODE>
__global__ void __launch_bounds__(256) k_probe_atomic(uint8_t *base, size_t stride, uint64_t sym_off, unsigned npes,
                                                      unsigned long long words, size_t n, unsigned long long *sink) {
    unsigned long long acc = 0;
    const size_t T = (size_t)gridDim.x * blockDim.x;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += T) {
        // uniform over npes x words without integer division (a 64-bit modulo would make the probe ALU-bound):
        // multiply-high of two independent halves of the hash
        const unsigned long long h = probe_hash(i);
        const unsigned pe = __umulhi((unsigned)h, npes);
        const unsigned long long wd = __umul64hi(h ^ (h << 32), words);
        unsigned long long *p = reinterpret_cast<unsigned long long *>(base + (size_t)pe * stride + sym_off) + wd;
        if (MODE == SHMEMG_PROBE_RED_ADD) {
            asm volatile("red.relaxed.gpu.global.add.u64 [%0], %1;" ::"l"(p), "l"(0ull) : "memory");
        } else if (MODE == SHMEMG_PROBE_ATOM_ADD) {
            acc ^= atomicAdd(p, 0ull);
        } else {
            acc ^= atomicCAS(p, 0x5DEECE66D1234567ull ^ h, 0ull);   // compare value the word never holds
        }
    }
    if (MODE != SHMEMG_PROBE_RED_ADD && acc == 0x0123456789ABCDEFull && n == (size_t)-1) *sink = acc;
}

// The same bare atomics on a GIVEN address stream (op i -> word elem_idx[i] of PE tgt_pe[i]: the workload's own operand
// arrays, 8 bytes read per op, nothing written) or on ONE address, with or without warp aggregation (one L2 atomic per
// distinct address and warp, as SHMEMG_AMO_WARP_AGGREGATE issues them): the like-for-like ceilings of SURVEY.md 8(d) (iii) / (iv).
template <int MODE, bool AGG, bool STREAM>
__global__ void __launch_bounds__(256) k_probe_atomic2(uint8_t *base, size_t stride, uint64_t sym_off, const int *tgt_pe,
                                                       const unsigned *elem_idx, size_t n, unsigned long long *sink) {
    unsigned long long acc = 0;
    const size_t T = (size_t)gridDim.x * blockDim.x;
    const int lane = threadIdx.x & 31;
    const size_t first = ((size_t)blockIdx.x * blockDim.x + threadIdx.x) - lane;
    for (size_t i0 = first; i0 < n; i0 += T) {                 // warp-uniform trip count (match.any below)
        const size_t i = i0 + lane;
        const bool ok = i < n;
        unsigned long long *p = reinterpret_cast<unsigned long long *>(base + sym_off);
        if (STREAM && ok) p = reinterpret_cast<unsigned long long *>(base + (size_t)tgt_pe[i] * stride + sym_off) + elem_idx[i];
        bool issue = ok;
        if (AGG) {
            const unsigned grp = __match_any_sync(0xffffffffu, ok ? (unsigned long long)p : (unsigned long long)lane);
            issue = ok && lane == __ffs(grp) - 1;
        }
        if (!issue) continue;
        if (MODE == SHMEMG_PROBE_RED_ADD) asm volatile("red.relaxed.gpu.global.add.u64 [%0], %1;" ::"l"(p), "l"(0ull) : "memory");
        else if (MODE == SHMEMG_PROBE_ATOM_ADD) acc ^= atomicAdd(p, 0ull);
        else acc ^= atomicCAS(p, 0x5DEECE66D1234567ull ^ (unsigned long long)i, 0ull);
    }
    if (MODE != SHMEMG_PROBE_RED_ADD && acc == 0x0123456789ABCDEFull && n == (size_t)-1) *sink = acc;
}

__global__ void __launch_bounds__(SHMEMG_THREADS, 4)
k_probe_copy_all(uint8_t *base, size_t stride, uint64_t dst_off, uint64_t src_off, size_t nbytes, unsigned npes,
                 unsigned chunk, unsigned chunks_per_pe) {
    const size_t nwork = (size_t)npes * chunks_per_pe;
    for (size_t wk = blockIdx.x; wk < nwork; wk += gridDim.x) {
        const unsigned p = (unsigned)(wk / chunks_per_pe), c = (unsigned)(wk % chunks_per_pe);
        const size_t off = (size_t)c * chunk;
        size_t m = nbytes - off;
        if (m > chunk) m = chunk;
        copy_coop<8>(base + (size_t)p * stride + dst_off + off, base + (size_t)p * stride + src_off + off, m, threadIdx.x,
                     SHMEMG_THREADS);
    }
}


__global__ void __launch_bounds__(32)
k_probe_copy_all_tma(uint8_t *base, size_t stride, uint64_t dst_off, uint64_t src_off, size_t nbytes, unsigned npes,
                     unsigned chunks_per_pe) {
    extern __shared__ __align__(1024) uint8_t stage[];
    __shared__ uint64_t full[SHMEMG_TMA_STAGES];
    if (threadIdx.x != 0) return;
    tma_stream_init(full);
    tma_stream_copy(stage, full, blockIdx.x, gridDim.x, (size_t)npes * chunks_per_pe,
                    [&](size_t wk, const uint8_t *&s, uint8_t *&d, unsigned &n) {
        const size_t p = wk / chunks_per_pe, off = (wk % chunks_per_pe) * (size_t)SHMEMG_TMA_TILE;
        n = (unsigned)(nbytes - off < SHMEMG_TMA_TILE ? nbytes - off : SHMEMG_TMA_TILE);
        s = base + p * stride + src_off + off;
        d = base + p * stride + dst_off + off;
    });
}

extern "C" int shmemg_probe_atomic_on_stream(shmemg_world_t *w, int mode, uint64_t sym_off, uint64_t words_per_pe,
                                             size_t n, void *stream) {
    if (!w || mode < SHMEMG_PROBE_RED_ADD || mode > SHMEMG_PROBE_ATOM_CAS || words_per_pe == 0) return SHMEMG_ERR_ARG;
    if (sym_off & 7) return SHMEMG_ERR_ALIGN;
    if (words_per_pe > (w->heap_bytes >> 3) || !shmemg_in_range(w, sym_off, words_per_pe * 8)) return SHMEMG_ERR_RANGE;
    if (n == 0) return SHMEMG_OK;
    size_t blocks = (n + 255) / 256;
    const size_t cap = (size_t)w->sm_count * 8 * 4;
    if (blocks > cap) blocks = cap;
    unsigned long long *sink = reinterpret_cast<unsigned long long *>(&w->ctl->pad[0]);
    cudaStream_t st = (cudaStream_t)stream;
    if (mode == SHMEMG_PROBE_RED_ADD)
        k_probe_atomic<SHMEMG_PROBE_RED_ADD><<<(unsigned)blocks, 256, 0, st>>>(w->base, w->stride, sym_off, (unsigned)w->npes, words_per_pe, n, sink);
    else if (mode == SHMEMG_PROBE_ATOM_ADD)
        k_probe_atomic<SHMEMG_PROBE_ATOM_ADD><<<(unsigned)blocks, 256, 0, st>>>(w->base, w->stride, sym_off, (unsigned)w->npes, words_per_pe, n, sink);
    else
        k_probe_atomic<SHMEMG_PROBE_ATOM_CAS><<<(unsigned)blocks, 256, 0, st>>>(w->base, w->stride, sym_off, (unsigned)w->npes, words_per_pe, n, sink);
    SHMEMG_CUDA(w, cudaGetLastError());
    return SHMEMG_OK;
}

template <int MODE> static void launch_probe2(bool agg, bool stream_src, unsigned blocks, cudaStream_t st, uint8_t *base, size_t stride,
                                              uint64_t sym_off, const int *tgt, const unsigned *idx, size_t n, unsigned long long *sink) {
    if (agg) { if (stream_src) k_probe_atomic2<MODE, true, true><<<blocks, 256, 0, st>>>(base, stride, sym_off, tgt, idx, n, sink);
               else k_probe_atomic2<MODE, true, false><<<blocks, 256, 0, st>>>(base, stride, sym_off, tgt, idx, n, sink); }
    else { if (stream_src) k_probe_atomic2<MODE, false, true><<<blocks, 256, 0, st>>>(base, stride, sym_off, tgt, idx, n, sink);
           else k_probe_atomic2<MODE, false, false><<<blocks, 256, 0, st>>>(base, stride, sym_off, tgt, idx, n, sink); }
}

extern "C" int shmemg_probe_atomic_stream_on_stream(shmemg_world_t *w, int mode, uint64_t sym_off, const int32_t *tgt_pe,
                                                    const uint32_t *elem_idx, size_t n, int aggregate, void *stream) {
    if (!w || mode < SHMEMG_PROBE_RED_ADD || mode > SHMEMG_PROBE_ATOM_CAS || ((tgt_pe == nullptr) != (elem_idx == nullptr))) return SHMEMG_ERR_ARG;
    if (sym_off & 7) return SHMEMG_ERR_ALIGN;
    if (!shmemg_in_range(w, sym_off, 8)) return SHMEMG_ERR_RANGE;
    if (n == 0) return SHMEMG_OK;
    size_t blocks = (n + 255) / 256;
    const size_t cap = (size_t)w->sm_count * 8 * 4;
    if (blocks > cap) blocks = cap;
    unsigned long long *sink = reinterpret_cast<unsigned long long *>(&w->ctl->pad[0]);
    cudaStream_t st = (cudaStream_t)stream;
    const bool src = tgt_pe != nullptr;
    if (mode == SHMEMG_PROBE_RED_ADD) launch_probe2<SHMEMG_PROBE_RED_ADD>(aggregate != 0, src, (unsigned)blocks, st, w->base, w->stride, sym_off, tgt_pe, elem_idx, n, sink);
    else if (mode == SHMEMG_PROBE_ATOM_ADD) launch_probe2<SHMEMG_PROBE_ATOM_ADD>(aggregate != 0, src, (unsigned)blocks, st, w->base, w->stride, sym_off, tgt_pe, elem_idx, n, sink);
    else launch_probe2<SHMEMG_PROBE_ATOM_CAS>(aggregate != 0, src, (unsigned)blocks, st, w->base, w->stride, sym_off, tgt_pe, elem_idx, n, sink);
    SHMEMG_CUDA(w, cudaGetLastError());
    return SHMEMG_OK;
}

extern "C" int shmemg_probe_copy_all_on_stream(shmemg_world_t *w, uint64_t dst_off, uint64_t src_off, size_t nbytes,
                                               void *stream) {
    if (!w) return SHMEMG_ERR_ARG;
    if (!shmemg_in_range(w, dst_off, nbytes) || !shmemg_in_range(w, src_off, nbytes)) return SHMEMG_ERR_RANGE;
    if (nbytes == 0) return SHMEMG_OK;
    if (dst_off < src_off + nbytes && src_off < dst_off + nbytes) return SHMEMG_ERR_OVERLAP;
    if (((dst_off | src_off | nbytes | w->stride) & 15) == 0 && !w->tile_bytes_override) {
        if (!w->smem_attr_probe) {
            SHMEMG_CUDA(w, cudaFuncSetAttribute(k_probe_copy_all_tma, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SHMEMG_TMA_SMEM));
            w->smem_attr_probe = true;
        }
        const unsigned cpp = (unsigned)((nbytes + SHMEMG_TMA_TILE - 1) / SHMEMG_TMA_TILE);
        const uint64_t nwork = (uint64_t)w->npes * cpp;
        const unsigned grid = (unsigned)(nwork < (uint64_t)w->sm_count ? nwork : (uint64_t)w->sm_count);
        k_probe_copy_all_tma<<<grid, 32, SHMEMG_TMA_SMEM, (cudaStream_t)stream>>>(w->base, w->stride, dst_off, src_off, nbytes,
                                                                                 (unsigned)w->npes, cpp);
        SHMEMG_CUDA(w, cudaGetLastError());
        return SHMEMG_OK;
    }
    const uint64_t maxgrid = (uint64_t)w->sm_count * w->ctas_per_sm;
    unsigned chunk = 65536;
    if (w->tile_bytes_override) chunk = (unsigned)w->tile_bytes_override;
    const unsigned cpp = (unsigned)((nbytes + chunk - 1) / chunk);
    const uint64_t nwork = (uint64_t)w->npes * cpp;
    const unsigned grid = (unsigned)(nwork < maxgrid ? nwork : maxgrid);
    k_probe_copy_all<<<grid, SHMEMG_THREADS, 0, (cudaStream_t)stream>>>(w->base, w->stride, dst_off, src_off, nbytes,
                                                                        (unsigned)w->npes, chunk, cpp);
    SHMEMG_CUDA(w, cudaGetLastError());
    return SHMEMG_OK;
}
