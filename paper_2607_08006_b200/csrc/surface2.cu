// surface2.cu -- the rest of the OpenSHMEM op surface on the same heaps: broadcast,
// the generic AMO set on 32/64-bit words (L361), block-strided put/get (OpenSHMEM 1.6 ibput/ibget), signal test (L392).
// General reductions live with sum_reduce in collectives.cu.  sm_100a only; shares nothing with oracle/.
#include "tma_stream.cuh"

static bool ranges_overlap2(uint64_t a, uint64_t b, uint64_t na, uint64_t nb) { return a < b + nb && b < a + na; }

// ---- broadcast ------------------------------------------------------------------------------------------------------
// bulk-copy path: work item = (<= 32 KiB chunk of the root's source, destination PE); consecutive items (one per CTA) share
// the chunk, which is read from HBM once and from L2 by the others.  HBM-write bound: N*nbytes written, nbytes read.
__global__ void __launch_bounds__(32)
k_broadcast_tma(uint8_t *base, size_t stride, uint64_t dst_off, uint64_t src_off, size_t nbytes, int npes, int root) {
    extern __shared__ __align__(1024) uint8_t stage[];
    __shared__ uint64_t full[SHMEMG_TMA_STAGES];
    if (threadIdx.x != 0) return;
    tma_stream_init(full);
    const size_t chunks = (nbytes + SHMEMG_TMA_TILE - 1) / SHMEMG_TMA_TILE;
    const uint8_t *src = base + (size_t)root * stride + src_off;
    tma_stream_copy(stage, full, blockIdx.x, gridDim.x, chunks * npes, [&](size_t k, const uint8_t *&s, uint8_t *&d, unsigned &n) {
        const size_t j = k % npes, off = (k / npes) * SHMEMG_TMA_TILE;
        s = src + off;
        d = base + j * stride + dst_off + off;
        n = (unsigned)(nbytes - off < SHMEMG_TMA_TILE ? nbytes - off : SHMEMG_TMA_TILE);
    });
}
// register path (any alignment): work item = (16 KiB chunk, destination PE)
__global__ void __launch_bounds__(SHMEMG_THREADS, 4)
k_broadcast_bytes(uint8_t *base, size_t stride, uint64_t dst_off, uint64_t src_off, size_t nbytes, int npes, int root) {
    const size_t CH = 16384, chunks = (nbytes + CH - 1) / CH;
    const uint8_t *src = base + (size_t)root * stride + src_off;
    for (size_t k = blockIdx.x; k < chunks * npes; k += gridDim.x) {
        const size_t j = k % npes, off = (k / npes) * CH;
        copy_coop<4>(base + j * stride + dst_off + off, src + off, nbytes - off < CH ? nbytes - off : CH, threadIdx.x,
                     SHMEMG_THREADS);
    }
}

extern "C" int shmemg_broadcast_on_stream(shmemg_world_t *w, uint64_t dest_off, uint64_t source_off, size_t nbytes,
                                          int root_pe, void *stream) {
    if (!w) return SHMEMG_ERR_ARG;
    if (!shmemg_pe_ok(w, root_pe)) return SHMEMG_ERR_PE;
    if (!shmemg_in_range(w, dest_off, nbytes) || !shmemg_in_range(w, source_off, nbytes)) return SHMEMG_ERR_RANGE;
    if (nbytes == 0) return SHMEMG_OK;
    if (ranges_overlap2(dest_off, source_off, nbytes, nbytes)) return SHMEMG_ERR_OVERLAP;
    cudaStream_t st = (cudaStream_t)stream;
    if (((dest_off | source_off | nbytes | w->stride) & 15) == 0 && !w->tile_bytes_override) {
        if (!w->smem_attr_bcast) {
            SHMEMG_CUDA(w, cudaFuncSetAttribute(k_broadcast_tma, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SHMEMG_TMA_SMEM));
            w->smem_attr_bcast = true;
        }
        const uint64_t items = (uint64_t)((nbytes + SHMEMG_TMA_TILE - 1) / SHMEMG_TMA_TILE) * w->npes;
        const unsigned grid = (unsigned)(items < (uint64_t)w->sm_count ? items : (uint64_t)w->sm_count);
        k_broadcast_tma<<<grid, 32, SHMEMG_TMA_SMEM, st>>>(w->base, w->stride, dest_off, source_off, nbytes, w->npes, root_pe);
    } else {
        const uint64_t items = (uint64_t)((nbytes + 16383) / 16384) * w->npes, maxgrid = (uint64_t)w->sm_count * w->ctas_per_sm;
        k_broadcast_bytes<<<(unsigned)(items < maxgrid ? items : maxgrid), SHMEMG_THREADS, 0, st>>>(w->base, w->stride, dest_off,
                                                                                                  source_off, nbytes, w->npes, root_pe);
    }
    SHMEMG_CUDA(w, cudaGetLastError());
    return SHMEMG_OK;
}

// ---- generic AMO batch ------------------------------------------------------------------------------------------------
// One op per thread and trip, 4 trips in flight.  red.global when nothing is fetched (st for SET), atom.global when the old
// value is returned (ld for FETCH): L2 atomic throughput is the bound, as for the add / fetch-add / compare-swap calls.
struct Amo2Args {
    uint8_t *base;
    size_t stride;
    uint64_t sym_off;
    const int *tgt_pe;
    const void *idx;
    const unsigned long long *val;
    unsigned long long val_s;
    unsigned long long *fetched;
    size_t n;
};

template <typename T, int OP, bool FETCH> __device__ __forceinline__ T amo2_one(T *word, T v) {
    if (OP == SHMEMG_AMO_FETCH) {                               // atomic read (a strong relaxed load at GPU scope)
        T r;
        if constexpr (sizeof(T) == 8) asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(r) : "l"(word) : "memory");
        else asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(r) : "l"(word) : "memory");
        return r;
    }
    if (FETCH) {
        switch (OP) {
        case SHMEMG_AMO_ADD: return atomicAdd(word, v);
        case SHMEMG_AMO_AND: return atomicAnd(word, v);
        case SHMEMG_AMO_OR: return atomicOr(word, v);
        case SHMEMG_AMO_XOR: return atomicXor(word, v);
        default: return atomicExch(word, v);
        }
    }
    if constexpr (sizeof(T) == 8) {
        switch (OP) {
        case SHMEMG_AMO_ADD: asm volatile("red.relaxed.gpu.global.add.u64 [%0], %1;" ::"l"(word), "l"(v) : "memory"); break;
        case SHMEMG_AMO_AND: asm volatile("red.relaxed.gpu.global.and.b64 [%0], %1;" ::"l"(word), "l"(v) : "memory"); break;
        case SHMEMG_AMO_OR: asm volatile("red.relaxed.gpu.global.or.b64 [%0], %1;" ::"l"(word), "l"(v) : "memory"); break;
        case SHMEMG_AMO_XOR: asm volatile("red.relaxed.gpu.global.xor.b64 [%0], %1;" ::"l"(word), "l"(v) : "memory"); break;
        default: asm volatile("st.relaxed.gpu.global.u64 [%0], %1;" ::"l"(word), "l"(v) : "memory"); break;   // atomic_set
        }
    } else {
        switch (OP) {
        case SHMEMG_AMO_ADD: asm volatile("red.relaxed.gpu.global.add.u32 [%0], %1;" ::"l"(word), "r"(v) : "memory"); break;
        case SHMEMG_AMO_AND: asm volatile("red.relaxed.gpu.global.and.b32 [%0], %1;" ::"l"(word), "r"(v) : "memory"); break;
        case SHMEMG_AMO_OR: asm volatile("red.relaxed.gpu.global.or.b32 [%0], %1;" ::"l"(word), "r"(v) : "memory"); break;
        case SHMEMG_AMO_XOR: asm volatile("red.relaxed.gpu.global.xor.b32 [%0], %1;" ::"l"(word), "r"(v) : "memory"); break;
        default: asm volatile("st.relaxed.gpu.global.u32 [%0], %1;" ::"l"(word), "r"(v) : "memory"); break;
        }
    }
    return 0;
}

template <typename T, int IDXB, int OP, bool FETCH>
__global__ void __launch_bounds__(256) k_amo2(const Amo2Args a) {
    const size_t T4 = (size_t)gridDim.x * blockDim.x;
    for (size_t i0 = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i0 < a.n; i0 += 4 * T4) {
        T *word[4];
        T v[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            const size_t i = i0 + (size_t)k * T4;
            word[k] = nullptr;
            if (i < a.n) {
                const unsigned long long e = IDXB == 4 ? (unsigned long long)reinterpret_cast<const unsigned *>(a.idx)[i]
                                                       : reinterpret_cast<const unsigned long long *>(a.idx)[i];
                word[k] = reinterpret_cast<T *>(a.base + (size_t)a.tgt_pe[i] * a.stride + a.sym_off) + e;
                v[k] = (T)(a.val ? a.val[i] : a.val_s);
            }
        }
        T old[4];
#pragma unroll
        for (int k = 0; k < 4; ++k)
            if (word[k]) old[k] = amo2_one<T, OP, FETCH>(word[k], v[k]);
        if (FETCH) {
#pragma unroll
            for (int k = 0; k < 4; ++k)
                if (word[k]) a.fetched[i0 + (size_t)k * T4] = (unsigned long long)old[k];
        }
    }
}

template <typename T, int IDXB, int OP> static void launch_amo2_f(const Amo2Args &a, unsigned blocks, cudaStream_t st) {
    if (a.fetched) k_amo2<T, IDXB, OP, true><<<blocks, 256, 0, st>>>(a);
    else k_amo2<T, IDXB, OP, false><<<blocks, 256, 0, st>>>(a);
}
template <typename T, int IDXB> static void launch_amo2_op(int op, const Amo2Args &a, unsigned blocks, cudaStream_t st) {
    switch (op) {
    case SHMEMG_AMO_ADD: launch_amo2_f<T, IDXB, SHMEMG_AMO_ADD>(a, blocks, st); break;
    case SHMEMG_AMO_AND: launch_amo2_f<T, IDXB, SHMEMG_AMO_AND>(a, blocks, st); break;
    case SHMEMG_AMO_OR: launch_amo2_f<T, IDXB, SHMEMG_AMO_OR>(a, blocks, st); break;
    case SHMEMG_AMO_XOR: launch_amo2_f<T, IDXB, SHMEMG_AMO_XOR>(a, blocks, st); break;
    case SHMEMG_AMO_SWAP: launch_amo2_f<T, IDXB, SHMEMG_AMO_SWAP>(a, blocks, st); break;
    default: k_amo2<T, IDXB, SHMEMG_AMO_FETCH, true><<<blocks, 256, 0, st>>>(a); break;
    }
}

extern "C" int shmemg_atomic_op_batch_on_stream(shmemg_world_t *w, int amo, int width, uint64_t sym_off,
                                                const int32_t *tgt_pe, const void *elem_idx, int idx_bytes,
                                                const uint64_t *val, uint64_t val_scalar, uint64_t *fetched_out,
                                                size_t n, void *stream) {
    if (!w || amo < SHMEMG_AMO_ADD || amo > SHMEMG_AMO_FETCH || (width != 4 && width != 8)) return SHMEMG_ERR_ARG;
    if (n && (!tgt_pe || !elem_idx)) return SHMEMG_ERR_ARG;
    if (idx_bytes != 4 && idx_bytes != 8) return SHMEMG_ERR_ARG;
    if (amo == SHMEMG_AMO_FETCH && n && !fetched_out) return SHMEMG_ERR_ARG;
    if (sym_off & (uint64_t)(width - 1)) return SHMEMG_ERR_ALIGN;
    if (!shmemg_in_range(w, sym_off, (uint64_t)width)) return SHMEMG_ERR_RANGE;
    if (n == 0) return SHMEMG_OK;
    // tgt_pe[] and elem_idx[] are DEVICE arrays: per-op bounds are the caller's contract (undefined otherwise)
    Amo2Args a{w->base, w->stride, sym_off, tgt_pe, elem_idx, (const unsigned long long *)val, val_scalar,
               (unsigned long long *)fetched_out, n};
    size_t blocks = (n + 1023) / 1024;
    const size_t cap = (size_t)w->sm_count * 8 * 4;
    if (blocks > cap) blocks = cap;
    cudaStream_t st = (cudaStream_t)stream;
    if (width == 8) {
        if (idx_bytes == 4) launch_amo2_op<unsigned long long, 4>(amo, a, (unsigned)blocks, st);
        else launch_amo2_op<unsigned long long, 8>(amo, a, (unsigned)blocks, st);
    } else {
        if (idx_bytes == 4) launch_amo2_op<unsigned, 4>(amo, a, (unsigned)blocks, st);
        else launch_amo2_op<unsigned, 8>(amo, a, (unsigned)blocks, st);
    }
    SHMEMG_CUDA(w, cudaGetLastError());
    return SHMEMG_OK;
}

// compare-swap on 4- or 8-byte words (the remaining AMO of the inherited set): atom.global.cas.b32 / .b64, four
// independent ops per thread in flight, fetched values written coalesced.
struct Cswap2Args {
    uint8_t *base;
    size_t stride;
    uint64_t sym_off;
    const int *tgt_pe;
    const void *idx;
    const unsigned long long *cond, *val;
    unsigned long long cond_s, val_s;
    unsigned long long *fetched;
    size_t n;
};
template <typename T, int IDXB>
__global__ void __launch_bounds__(256) k_cswap2(const Cswap2Args a) {
    const size_t T4 = (size_t)gridDim.x * blockDim.x;
    for (size_t i0 = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i0 < a.n; i0 += 4 * T4) {
        T *word[4];
        T c[4], v[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            const size_t i = i0 + (size_t)k * T4;
            word[k] = nullptr;
            if (i < a.n) {
                const unsigned long long e = IDXB == 4 ? (unsigned long long)reinterpret_cast<const unsigned *>(a.idx)[i]
                                                       : reinterpret_cast<const unsigned long long *>(a.idx)[i];
                word[k] = reinterpret_cast<T *>(a.base + (size_t)a.tgt_pe[i] * a.stride + a.sym_off) + e;
                c[k] = (T)(a.cond ? a.cond[i] : a.cond_s);
                v[k] = (T)(a.val ? a.val[i] : a.val_s);
            }
        }
        T old[4];
#pragma unroll
        for (int k = 0; k < 4; ++k)
            if (word[k]) old[k] = atomicCAS(word[k], c[k], v[k]);
#pragma unroll
        for (int k = 0; k < 4; ++k)
            if (word[k]) a.fetched[i0 + (size_t)k * T4] = (unsigned long long)old[k];
    }
}

extern "C" int shmemg_atomic_cswap_op_batch_on_stream(shmemg_world_t *w, int width, uint64_t sym_off, const int32_t *tgt_pe,
                                                      const void *elem_idx, int idx_bytes, const uint64_t *cond,
                                                      uint64_t cond_scalar, const uint64_t *val, uint64_t val_scalar,
                                                      uint64_t *fetched_out, size_t n, void *stream) {
    if (!w || (width != 4 && width != 8)) return SHMEMG_ERR_ARG;
    if (n && (!tgt_pe || !elem_idx || !fetched_out)) return SHMEMG_ERR_ARG;
    if (idx_bytes != 4 && idx_bytes != 8) return SHMEMG_ERR_ARG;
    if (sym_off & (uint64_t)(width - 1)) return SHMEMG_ERR_ALIGN;
    if (!shmemg_in_range(w, sym_off, (uint64_t)width)) return SHMEMG_ERR_RANGE;
    if (n == 0) return SHMEMG_OK;
    // tgt_pe[] and elem_idx[] are DEVICE arrays: per-op bounds are the caller's contract (undefined otherwise)
    Cswap2Args a{w->base, w->stride, sym_off, tgt_pe, elem_idx, (const unsigned long long *)cond, (const unsigned long long *)val,
                 cond_scalar, val_scalar, (unsigned long long *)fetched_out, n};
    size_t blocks = (n + 1023) / 1024;
    const size_t cap = (size_t)w->sm_count * 8 * 4;
    if (blocks > cap) blocks = cap;
    cudaStream_t st = (cudaStream_t)stream;
    if (width == 8) {
        if (idx_bytes == 4) k_cswap2<unsigned long long, 4><<<(unsigned)blocks, 256, 0, st>>>(a);
        else k_cswap2<unsigned long long, 8><<<(unsigned)blocks, 256, 0, st>>>(a);
    } else {
        if (idx_bytes == 4) k_cswap2<unsigned, 4><<<(unsigned)blocks, 256, 0, st>>>(a);
        else k_cswap2<unsigned, 8><<<(unsigned)blocks, 256, 0, st>>>(a);
    }
    SHMEMG_CUDA(w, cudaGetLastError());
    return SHMEMG_OK;
}

// Debug aid for the structure-of-arrays AMO calls: their tgt_pe[] / elem_idx[] live in DEVICE memory, so the host-side argument
// checks cannot see them and an out-of-range entry is a stray atomic somewhere in (or beyond) the slab.  This kernel reads the
// two arrays the way the AMO kernels do and records the smallest op index whose target word is not inside its PE's window.
template <int IDXB>
__global__ void __launch_bounds__(256) k_amo_check(const int *tgt_pe, const void *idx, size_t n, int npes, unsigned long long first_word,
                                                   unsigned long long words_in_window, unsigned long long *first_bad) {
    unsigned long long bad = ~0ull;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        const unsigned long long e = IDXB == 4 ? (unsigned long long)reinterpret_cast<const unsigned *>(idx)[i]
                                               : reinterpret_cast<const unsigned long long *>(idx)[i];
        const int t = tgt_pe[i];
        if ((t < 0 || t >= npes || e >= words_in_window - first_word) && i < bad) bad = i;      // first_word < words_in_window (host check)
    }
    if (bad != ~0ull) atomicMin(first_bad, bad);
}

extern "C" int shmemg_amo_check_batch_on_stream(shmemg_world_t *w, int width, uint64_t sym_off, const int32_t *tgt_pe,
                                                const void *elem_idx, int idx_bytes, size_t n, uint64_t *first_bad_dev,
                                                void *stream) {
    if (!w || (width != 4 && width != 8) || !first_bad_dev) return SHMEMG_ERR_ARG;
    if (n && (!tgt_pe || !elem_idx)) return SHMEMG_ERR_ARG;
    if (idx_bytes != 4 && idx_bytes != 8) return SHMEMG_ERR_ARG;
    if (sym_off & (uint64_t)(width - 1)) return SHMEMG_ERR_ALIGN;
    if (!shmemg_in_range(w, sym_off, (uint64_t)width)) return SHMEMG_ERR_RANGE;
    cudaStream_t st = (cudaStream_t)stream;
    SHMEMG_CUDA(w, cudaMemsetAsync(first_bad_dev, 0xff, 8, st));
    if (n == 0) return SHMEMG_OK;
    size_t blocks = (n + 255) / 256;
    const size_t cap = (size_t)w->sm_count * 8;
    if (blocks > cap) blocks = cap;
    const unsigned long long first_word = sym_off / (uint64_t)width, words = w->heap_bytes / (uint64_t)width;   // whole words of the window
    if (idx_bytes == 4) k_amo_check<4><<<(unsigned)blocks, 256, 0, st>>>(tgt_pe, elem_idx, n, w->npes, first_word, words, (unsigned long long *)first_bad_dev);
    else k_amo_check<8><<<(unsigned)blocks, 256, 0, st>>>(tgt_pe, elem_idx, n, w->npes, first_word, words, (unsigned long long *)first_bad_dev);
    SHMEMG_CUDA(w, cudaGetLastError());
    return SHMEMG_OK;
}

// ---- block-strided put / get --------------------------------------------------------------------------------------------
// Three paths, picked on the host:
//   bulk    blocks >= 1 KiB with 16-byte aligned addresses, strides and size: work item = (block, <= 32 KiB chunk), the
//           bulk-copy pipeline of put/get (a y-face of the halo cube is 256 blocks of 2 KiB);
//   element blocks of 4 / 8 / 16 naturally aligned bytes: one element per thread, so the contiguous side is coalesced and the
//           strided side costs one 32-byte sector per element (a z-face of the halo cube: stride 2 KiB);
//   generic anything else: one warp per block through the any-alignment cooperative copy.
__global__ void __launch_bounds__(32)
k_ib_tma(uint8_t *dst, const uint8_t *src, size_t dst_stride, size_t src_stride, size_t block, size_t nblocks) {
    extern __shared__ __align__(1024) uint8_t stage[];
    __shared__ uint64_t full[SHMEMG_TMA_STAGES];
    if (threadIdx.x != 0) return;
    tma_stream_init(full);
    const size_t cpb = (block + SHMEMG_TMA_TILE - 1) / SHMEMG_TMA_TILE;
    tma_stream_copy(stage, full, blockIdx.x, gridDim.x, nblocks * cpb, [&](size_t k, const uint8_t *&s, uint8_t *&d, unsigned &n) {
        const size_t b = k / cpb, off = (k % cpb) * SHMEMG_TMA_TILE;
        s = src + b * src_stride + off;
        d = dst + b * dst_stride + off;
        n = (unsigned)(block - off < SHMEMG_TMA_TILE ? block - off : SHMEMG_TMA_TILE);
    });
}
template <typename T>
__global__ void __launch_bounds__(256) k_ib_elem(uint8_t *dst, const uint8_t *src, size_t dst_stride, size_t src_stride,
                                                 size_t nblocks) {
    const size_t T4 = (size_t)gridDim.x * blockDim.x;
    for (size_t b0 = (size_t)blockIdx.x * blockDim.x + threadIdx.x; b0 < nblocks; b0 += 4 * T4) {
        T v[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            const size_t b = b0 + (size_t)k * T4;
            if (b < nblocks) v[k] = *reinterpret_cast<const volatile T *>(src + b * src_stride);
        }
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            const size_t b = b0 + (size_t)k * T4;
            if (b < nblocks) *reinterpret_cast<T *>(dst + b * dst_stride) = v[k];
        }
    }
}
struct Elem16 { unsigned long long a, b; };
template <>
__global__ void __launch_bounds__(256) k_ib_elem<Elem16>(uint8_t *dst, const uint8_t *src, size_t dst_stride, size_t src_stride,
                                                        size_t nblocks) {
    for (size_t b = (size_t)blockIdx.x * blockDim.x + threadIdx.x; b < nblocks; b += (size_t)gridDim.x * blockDim.x)
        st_stream16(dst + b * dst_stride, ld_stream16(src + b * src_stride));
}
__global__ void __launch_bounds__(256) k_ib_generic(uint8_t *dst, const uint8_t *src, size_t dst_stride, size_t src_stride,
                                                    size_t block, size_t nblocks) {
    const size_t warp = ((size_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5, nwarps = ((size_t)gridDim.x * blockDim.x) >> 5;
    for (size_t b = warp; b < nblocks; b += nwarps)
        copy_coop<2>(dst + b * dst_stride, src + b * src_stride, block, threadIdx.x & 31, 32);
}

static int launch_ib(shmemg_world *w, uint64_t dest_off, uint64_t source_off, uint64_t dst_stride, uint64_t src_stride,
                     size_t block, size_t nblocks, int dst_pe, int src_pe, cudaStream_t st) {
    if (block == 0 || nblocks == 0) return SHMEMG_OK;
    const uint64_t dspan = (uint64_t)(nblocks - 1) * dst_stride + block, sspan = (uint64_t)(nblocks - 1) * src_stride + block;
    if (dst_stride && (dspan - block) / dst_stride != nblocks - 1) return SHMEMG_ERR_RANGE;       // overflow
    if (src_stride && (sspan - block) / src_stride != nblocks - 1) return SHMEMG_ERR_RANGE;
    if (!shmemg_in_range(w, dest_off, dspan) || !shmemg_in_range(w, source_off, sspan)) return SHMEMG_ERR_RANGE;
    if (nblocks > 1 && dst_stride < block) return SHMEMG_ERR_OVERLAP;      // destination blocks would overlap each other
    uint8_t *dst = shmemg_addr(w, dst_pe, dest_off);
    const uint8_t *src = shmemg_addr(w, src_pe, source_off);
    const uint64_t all = (uint64_t)(uintptr_t)dst | (uint64_t)(uintptr_t)src | dst_stride | src_stride | block;
    const uint64_t maxgrid = (uint64_t)w->sm_count * 8;
    if (block >= 1024 && (all & 15) == 0) {
        if (!w->smem_attr_ib) {
            SHMEMG_CUDA(w, cudaFuncSetAttribute(k_ib_tma, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SHMEMG_TMA_SMEM));
            w->smem_attr_ib = true;
        }
        const uint64_t items = (uint64_t)nblocks * ((block + SHMEMG_TMA_TILE - 1) / SHMEMG_TMA_TILE);
        k_ib_tma<<<(unsigned)(items < (uint64_t)w->sm_count ? items : (uint64_t)w->sm_count), 32, SHMEMG_TMA_SMEM, st>>>(
            dst, src, dst_stride, src_stride, block, nblocks);
    } else if ((block == 4 || block == 8 || block == 16) && (all & (block - 1)) == 0) {
        uint64_t blocks = (nblocks + 1023) / 1024;
        if (blocks > maxgrid) blocks = maxgrid;
        if (block == 4) k_ib_elem<unsigned><<<(unsigned)blocks, 256, 0, st>>>(dst, src, dst_stride, src_stride, nblocks);
        else if (block == 8) k_ib_elem<unsigned long long><<<(unsigned)blocks, 256, 0, st>>>(dst, src, dst_stride, src_stride, nblocks);
        else k_ib_elem<Elem16><<<(unsigned)((nblocks + 255) / 256 < maxgrid ? (nblocks + 255) / 256 : maxgrid), 256, 0, st>>>(
                 dst, src, dst_stride, src_stride, nblocks);
    } else {
        uint64_t blocks = (nblocks + 7) / 8;
        if (blocks > maxgrid) blocks = maxgrid;
        k_ib_generic<<<(unsigned)blocks, 256, 0, st>>>(dst, src, dst_stride, src_stride, block, nblocks);
    }
    SHMEMG_CUDA(w, cudaGetLastError());
    return SHMEMG_OK;
}

extern "C" int shmemg_ibput_on_stream(shmemg_world_t *w, uint64_t dest_off, uint64_t source_off, uint64_t dst_stride,
                                      uint64_t src_stride, size_t block_bytes, size_t nblocks, int pe, int target_pe,
                                      void *stream) {
    if (!w) return SHMEMG_ERR_ARG;
    if (!shmemg_pe_ok(w, pe) || !shmemg_pe_ok(w, target_pe)) return SHMEMG_ERR_PE;
    return launch_ib(w, dest_off, source_off, dst_stride, src_stride, block_bytes, nblocks, target_pe, pe, (cudaStream_t)stream);
}
extern "C" int shmemg_ibget_on_stream(shmemg_world_t *w, uint64_t dest_off, uint64_t source_off, uint64_t dst_stride,
                                      uint64_t src_stride, size_t block_bytes, size_t nblocks, int pe, int target_pe,
                                      void *stream) {
    if (!w) return SHMEMG_ERR_ARG;
    if (!shmemg_pe_ok(w, pe) || !shmemg_pe_ok(w, target_pe)) return SHMEMG_ERR_PE;
    return launch_ib(w, dest_off, source_off, dst_stride, src_stride, block_bytes, nblocks, pe, target_pe, (cudaStream_t)stream);
}

// ---- signal test ------------------------------------------------------------------------------------------------------------
__global__ void k_signal_test(const unsigned long long *sig, int cmp, unsigned long long value, int *result) {
    const bool ok = cmp_u64(cmp, ld_relaxed_u64(sig), value);
    if (ok) fence_acquire();
    *result = ok ? 1 : 0;
}

extern "C" int shmemg_signal_test_on_stream(shmemg_world_t *w, uint64_t sig_off, int cmp, uint64_t value, int pe,
                                            int32_t *result_dev, void *stream) {
    if (!w || !result_dev || cmp < SHMEMG_CMP_EQ || cmp > SHMEMG_CMP_LE) return SHMEMG_ERR_ARG;
    if (!shmemg_pe_ok(w, pe)) return SHMEMG_ERR_PE;
    if (!shmemg_in_range(w, sig_off, 8)) return SHMEMG_ERR_RANGE;
    if (sig_off & 7) return SHMEMG_ERR_ALIGN;
    k_signal_test<<<1, 1, 0, (cudaStream_t)stream>>>(reinterpret_cast<const unsigned long long *>(shmemg_addr(w, pe, sig_off)), cmp,
                                                     value, result_dev);
    SHMEMG_CUDA(w, cudaGetLastError());
    return SHMEMG_OK;
}

// ---- teams (NEXT-3) -------------------------------------------------------------------------------------------------------
// A team is a strided set of PEs; member k's window is base + (start + k*stride) * heap_stride, i.e. the team is itself a
// "world" with base' = base + start*heap_stride, heap_stride' = stride*heap_stride, npes' = size.  The team collectives run the
// world entry points on that view (the fields are swapped for the duration of the enqueue; kernels take them by value).
static bool team_lookup(const shmemg_world *w, int team, shmemg_world::Team &t) {
    if (team == SHMEM_TEAM_WORLD || team == SHMEM_DEVICE_TEAM_WORLD || team == SHMEM_DEVICE_TEAM_SHARED) {
        t = {0, 1, w->teams_world_npes ? w->teams_world_npes : w->npes};
        return true;
    }
    if (team < SHMEMG_TEAM_USER0 || (size_t)(team - SHMEMG_TEAM_USER0) >= w->teams.size()) return false;
    t = w->teams[team - SHMEMG_TEAM_USER0];
    return true;
}
struct TeamView {
    shmemg_world *w;
    uint8_t *base; size_t stride; int npes;
    TeamView(shmemg_world *w_, const shmemg_world::Team &t) : w(w_), base(w_->base), stride(w_->stride), npes(w_->npes) {
        w->teams_world_npes = npes;
        w->base = base + (size_t)t.start * stride;
        w->stride = stride * (size_t)t.stride;
        w->npes = t.size;
    }
    ~TeamView() { w->base = base; w->stride = stride; w->npes = npes; w->teams_world_npes = 0; }
};

extern "C" int shmemg_team_split_strided(shmemg_world_t *w, int parent_team, int start, int stride, int size, int *new_team) {
    if (!w || !new_team) return SHMEMG_ERR_ARG;
    shmemg_world::Team p;
    if (!team_lookup(w, parent_team, p)) return SHMEMG_ERR_ARG;
    if (size < 1 || stride < 1 || start < 0 || (long long)start + (long long)(size - 1) * stride >= p.size) return SHMEMG_ERR_PE;
    w->teams.push_back({p.start + start * p.stride, p.stride * stride, size});
    *new_team = SHMEMG_TEAM_USER0 + (int)w->teams.size() - 1;
    return SHMEMG_OK;
}
extern "C" int shmemg_team_n_pes(const shmemg_world_t *w, int team) {
    shmemg_world::Team t;
    return (w && team_lookup(w, team, t)) ? t.size : SHMEMG_ERR_ARG;
}
extern "C" int shmemg_team_translate_pe(const shmemg_world_t *w, int team, int rank) {
    shmemg_world::Team t;
    if (!w || !team_lookup(w, team, t)) return SHMEMG_ERR_ARG;
    return (rank >= 0 && rank < t.size) ? t.start + rank * t.stride : SHMEMG_ERR_PE;
}
#define TEAM_CALL(call)                                        \
    shmemg_world::Team t;                                      \
    if (!w || !team_lookup(w, team, t)) return SHMEMG_ERR_ARG; \
    TeamView view(w, t);                                       \
    return call;
extern "C" int shmemg_team_reduce_on_stream(shmemg_world_t *w, int team, int op, int dtype, uint64_t dest_off,
                                            uint64_t source_off, size_t nreduce, void *stream) {
    TEAM_CALL(shmemg_reduce_on_stream(w, op, dtype, dest_off, source_off, nreduce, stream))
}
extern "C" int shmemg_team_fcollect_on_stream(shmemg_world_t *w, int team, uint64_t dest_off, uint64_t source_off,
                                              size_t nbytes, void *stream) {
    TEAM_CALL(shmemg_fcollect_on_stream(w, dest_off, source_off, nbytes, stream))
}
extern "C" int shmemg_team_alltoall_on_stream(shmemg_world_t *w, int team, uint64_t dest_off, uint64_t source_off,
                                              size_t nbytes, void *stream) {
    TEAM_CALL(shmemg_alltoall_on_stream(w, dest_off, source_off, nbytes, stream))
}
extern "C" int shmemg_team_broadcast_on_stream(shmemg_world_t *w, int team, uint64_t dest_off, uint64_t source_off,
                                               size_t nbytes, int root_rank, void *stream) {
    TEAM_CALL(shmemg_broadcast_on_stream(w, dest_off, source_off, nbytes, root_rank, stream))
}

// ---- vector test / wait (OpenSHMEM 1.6 test_all / any / some and wait_until_all / any / some) -----------------
// One block; thread t looks at words t, t + 256, ...  `wait`: the block polls until the mode's condition holds (all words /
// at least one word).  Then thread 0 lists the satisfied positions in ascending order (at least the ones that made the
// condition true; a word that becomes true in between is a legitimate member too) into indices_dev and their number into
// count_dev (either may be NULL).  A satisfied result is an acquire.
__global__ void __launch_bounds__(256) k_signal_vec(const unsigned long long *sig, size_t nelems, int cmp, unsigned long long value,
                                                    int need_all, int wait, unsigned long long *indices, unsigned long long *count) {
    for (;;) {
        int ok_all = 1, ok_any = 0;
        for (size_t k = threadIdx.x; k < nelems; k += blockDim.x) {
            const bool ok = cmp_u64(cmp, ld_relaxed_u64(sig + k), value);
            ok_all &= ok; ok_any |= ok;
        }
        const int all = __syncthreads_and(ok_all), any = __syncthreads_or(ok_any);
        if (!wait || nelems == 0 || (need_all ? all : any)) break;
        __nanosleep(64);
    }
    fence_acquire();
    if (threadIdx.x == 0) {
        unsigned long long n = 0;
        for (size_t k = 0; k < nelems; ++k)
            if (cmp_u64(cmp, ld_relaxed_u64(sig + k), value)) { if (indices) indices[n] = k; ++n; }
        fence_acquire();
        if (count) *count = n;
    }
}

static int signal_vec(shmemg_world_t *w, uint64_t sig_off, size_t nelems, int cmp, uint64_t value, int pe, int need_all, int wait,
                      uint64_t *indices_dev, uint64_t *count_dev, void *stream) {
    if (!w || cmp < SHMEMG_CMP_EQ || cmp > SHMEMG_CMP_LE) return SHMEMG_ERR_ARG;
    if (!shmemg_pe_ok(w, pe)) return SHMEMG_ERR_PE;
    if (nelems > (SIZE_MAX >> 3) || !shmemg_in_range(w, sig_off, 8 * (uint64_t)nelems)) return SHMEMG_ERR_RANGE;
    if (sig_off & 7) return SHMEMG_ERR_ALIGN;
    k_signal_vec<<<1, 256, 0, (cudaStream_t)stream>>>(reinterpret_cast<const unsigned long long *>(shmemg_addr(w, pe, sig_off)), nelems,
                                                     cmp, value, need_all, wait, (unsigned long long *)indices_dev,
                                                     (unsigned long long *)count_dev);
    SHMEMG_CUDA(w, cudaGetLastError());
    return SHMEMG_OK;
}
extern "C" int shmemg_signal_test_vec_on_stream(shmemg_world_t *w, uint64_t sig_off, size_t nelems, int cmp, uint64_t value, int pe,
                                                uint64_t *indices_dev, uint64_t *count_dev, void *stream) {
    return signal_vec(w, sig_off, nelems, cmp, value, pe, 0, 0, indices_dev, count_dev, stream);
}
extern "C" int shmemg_signal_wait_until_all_on_stream(shmemg_world_t *w, uint64_t sig_off, size_t nelems, int cmp, uint64_t value,
                                                      int pe, void *stream) {
    return signal_vec(w, sig_off, nelems, cmp, value, pe, 1, 1, nullptr, nullptr, stream);
}
extern "C" int shmemg_signal_wait_until_some_on_stream(shmemg_world_t *w, uint64_t sig_off, size_t nelems, int cmp, uint64_t value,
                                                       int pe, uint64_t *indices_dev, uint64_t *count_dev, void *stream) {
    return signal_vec(w, sig_off, nelems, cmp, value, pe, 0, 1, indices_dev, count_dev, stream);
}
