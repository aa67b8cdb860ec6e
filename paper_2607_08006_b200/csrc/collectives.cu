// collectives.cu -- world-team collectives, one kernel each.
//   alltoall   : tiled transpose-copy, 128-bit streaming accesses; HBM-bound, 2*N*N*blk bytes
//   fcollect   : each source chunk is read once into registers and stored to all N destinations (write-bound)
//   sum_reduce : bulk-copy pipeline per column tile: N windows streamed through shared memory, fp64 accumulation for
//                fp32 in ascending PE order, N-way replicated bulk store
//   barrier    : stream-level (kernel boundary) and in-kernel (one CTA per PE, cooperative launch)
#include "tma_stream.cuh"

// ---- alltoall: PE j's dest block i = PE i's source block j -------------------------------------------------------
__global__ void __launch_bounds__(SHMEMG_THREADS, 4)
k_alltoall(uint8_t *base, size_t stride, uint64_t dst_off, uint64_t src_off, size_t blk, int npes, unsigned chunk,
           unsigned chunks_per_blk) {
    const size_t nwork = (size_t)npes * npes * chunks_per_blk;
    for (size_t wk = blockIdx.x; wk < nwork; wk += gridDim.x) {
        const unsigned c = (unsigned)(wk % chunks_per_blk);
        const size_t ij = wk / chunks_per_blk;
        const int j = (int)(ij % npes), i = (int)(ij / npes);        // source-major: PE i's row is read contiguously
        const size_t off = (size_t)c * chunk;
        size_t n = blk - off;
        if (n > chunk) n = chunk;
        copy_coop<8>(base + (size_t)j * stride + dst_off + (size_t)i * blk + off,
                     base + (size_t)i * stride + src_off + (size_t)j * blk + off, n, threadIdx.x, SHMEMG_THREADS);
    }
}


// bulk-copy path (block size, offsets and stride 16-byte aligned): one issuing thread per CTA, work item =
// (source PE i, destination PE j, <= 32 KiB chunk), source-major so each CTA streams one PE's row
__global__ void __launch_bounds__(32)
k_alltoall_tma(uint8_t *base, size_t stride, uint64_t dst_off, uint64_t src_off, size_t blk, int npes, unsigned chunks_per_blk) {
    extern __shared__ __align__(1024) uint8_t stage[];
    __shared__ uint64_t full[SHMEMG_TMA_STAGES];
    if (threadIdx.x != 0) return;
    tma_stream_init(full);
    const size_t nwork = (size_t)npes * npes * chunks_per_blk;
    tma_stream_copy(stage, full, blockIdx.x, gridDim.x, nwork, [&](size_t wk, const uint8_t *&s, uint8_t *&d, unsigned &n) {
        const unsigned c = (unsigned)(wk % chunks_per_blk);
        const size_t ij = wk / chunks_per_blk;
        const int j = (int)(ij % npes), i = (int)(ij / npes);
        const size_t off = (size_t)c * SHMEMG_TMA_TILE;
        n = (unsigned)(blk - off < SHMEMG_TMA_TILE ? blk - off : SHMEMG_TMA_TILE);
        s = base + (size_t)i * stride + src_off + (size_t)j * blk + off;
        d = base + (size_t)j * stride + dst_off + (size_t)i * blk + off;
    });
}

// ---- block-strided alltoall (NEXT-4 (i): FFT-style transposes) --------------------------------------------------
// PE j's dest[i*dps + b*dbs .. +blk) = PE i's source[j*sps + b*sbs .. +blk).  Work items are ordered (source PE i, block b,
// destination PE j, chunk): for a slab transpose the chunks of consecutive j are contiguous in the source, so every CTA streams
// its share of the source like a plain copy and scatters 32 KiB pieces over the destination windows.
struct A2asArgs {
    uint8_t *base;
    size_t stride;
    uint64_t dst_off, src_off, dps, sps, dbs, sbs, blk, nblocks;
    int npes;
};
__global__ void __launch_bounds__(32) k_alltoalls_tma(const A2asArgs a, unsigned cpb) {
    extern __shared__ __align__(1024) uint8_t stage[];
    __shared__ uint64_t full[SHMEMG_TMA_STAGES];
    if (threadIdx.x != 0) return;
    tma_stream_init(full);
    const size_t nwork = (size_t)a.npes * a.nblocks * a.npes * cpb;
    tma_stream_copy(stage, full, blockIdx.x, gridDim.x, nwork, [&](size_t wk, const uint8_t *&s, uint8_t *&d, unsigned &n) {
        const unsigned c = (unsigned)(wk % cpb);
        size_t r = wk / cpb;
        const size_t j = r % a.npes; r /= a.npes;
        const size_t b = r % a.nblocks, i = r / a.nblocks;
        const size_t off = (size_t)c * SHMEMG_TMA_TILE;
        n = (unsigned)(a.blk - off < SHMEMG_TMA_TILE ? a.blk - off : SHMEMG_TMA_TILE);
        s = a.base + i * a.stride + a.src_off + j * a.sps + b * a.sbs + off;
        d = a.base + j * a.stride + a.dst_off + i * a.dps + b * a.dbs + off;
    });
}
// any alignment: one CTA per (i, b, j, 16 KiB chunk)
__global__ void __launch_bounds__(SHMEMG_THREADS, 4) k_alltoalls_generic(const A2asArgs a, unsigned cpb) {
    const size_t nwork = (size_t)a.npes * a.nblocks * a.npes * cpb;
    for (size_t wk = blockIdx.x; wk < nwork; wk += gridDim.x) {
        const unsigned c = (unsigned)(wk % cpb);
        size_t r = wk / cpb;
        const size_t j = r % a.npes; r /= a.npes;
        const size_t b = r % a.nblocks, i = r / a.nblocks;
        const size_t off = (size_t)c * 16384;
        const size_t n = a.blk - off < 16384 ? a.blk - off : 16384;
        copy_coop<4>(a.base + j * a.stride + a.dst_off + i * a.dps + b * a.dbs + off,
                     a.base + i * a.stride + a.src_off + j * a.sps + b * a.sbs + off, n, threadIdx.x, SHMEMG_THREADS);
    }
}
// naturally aligned elements of 4 / 8 / 16 bytes (the OpenSHMEM alltoalls form): one element per thread; consecutive threads
// take consecutive blocks b of one (i, j) pair
template <typename T>
__global__ void __launch_bounds__(256) k_alltoalls_elem(const A2asArgs a) {
    const size_t n = (size_t)a.npes * a.npes * a.nblocks;
    for (size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x; e < n; e += (size_t)gridDim.x * blockDim.x) {
        const size_t b = e % a.nblocks, ij = e / a.nblocks, j = ij % a.npes, i = ij / a.npes;
        uint8_t *d = a.base + j * a.stride + a.dst_off + i * a.dps + b * a.dbs;
        const uint8_t *s = a.base + i * a.stride + a.src_off + j * a.sps + b * a.sbs;
        if constexpr (sizeof(T) == 16) st_stream16(d, ld_stream16(s));
        else *reinterpret_cast<T *>(d) = *reinterpret_cast<const volatile T *>(s);
    }
}

// ---- fcollect: PE j's dest[p*n .. +n) = PE p's source[0 .. n) for every j -------------------------------------------
// work item = (source PE p, 16-byte-vector chunk of its block, group of destination PEs)
template <int VPT>   // vectors per thread held in registers
__global__ void __launch_bounds__(SHMEMG_THREADS, 4)
k_fcollect_vec(uint8_t *base, size_t stride, uint64_t dst_off, uint64_t src_off, size_t nbytes, int npes,
               unsigned chunks_per_blk, int dst_groups) {
    const size_t nvec = nbytes >> 4;
    const unsigned chunk_vecs = SHMEMG_THREADS * VPT;
    const size_t nwork = (size_t)npes * chunks_per_blk * dst_groups;
    const int per_group = (npes + dst_groups - 1) / dst_groups;
    for (size_t wk = blockIdx.x; wk < nwork; wk += gridDim.x) {
        const int g = (int)(wk % dst_groups);
        const size_t pc = wk / dst_groups;
        const unsigned c = (unsigned)(pc % chunks_per_blk);
        const int p = (int)(pc / chunks_per_blk);
        const int4 *s = reinterpret_cast<const int4 *>(base + (size_t)p * stride + src_off) + (size_t)c * chunk_vecs;
        const size_t left = nvec - (size_t)c * chunk_vecs;
        int4 v[VPT];
#pragma unroll
        for (int u = 0; u < VPT; ++u) {
            const size_t k = threadIdx.x + (size_t)u * SHMEMG_THREADS;
            if (k < left) v[u] = ld_stream16(s + k);
        }
        const int j0 = g * per_group, j1 = min(npes, j0 + per_group);
        for (int j = j0; j < j1; ++j) {
            int4 *d = reinterpret_cast<int4 *>(base + (size_t)j * stride + dst_off + (size_t)p * nbytes) + (size_t)c * chunk_vecs;
#pragma unroll
            for (int u = 0; u < VPT; ++u) {
                const size_t k = threadIdx.x + (size_t)u * SHMEMG_THREADS;
                if (k < left) st_stream16(d + k, v[u]);
            }
        }
    }
}

// bulk-copy path: each work item (source PE p, <= 32 KiB chunk, group of destination PEs) is loaded into shared memory
// ONCE and stored from there to every destination of the group; the source (N x nbytes) is read from HBM once and
// from L2 by the other groups.  One issuing thread per CTA; STAGES-1 loads in flight ahead of the store front.
__global__ void __launch_bounds__(32)
k_fcollect_tma(uint8_t *base, size_t stride, uint64_t dst_off, uint64_t src_off, size_t nbytes, int npes,
               unsigned chunks_per_blk, int dst_groups) {
    extern __shared__ __align__(1024) uint8_t stage[];
    __shared__ uint64_t full[SHMEMG_TMA_STAGES];
    if (threadIdx.x != 0) return;
    tma_stream_init(full);
    const size_t nwork = (size_t)npes * chunks_per_blk * dst_groups;
    const int per_group = (npes + dst_groups - 1) / dst_groups;
    const size_t first = blockIdx.x, step = gridDim.x;
    const size_t mine = first < nwork ? (nwork - first + step - 1) / step : 0;
    auto decode = [&](size_t it, int &p, int &g, size_t &off, unsigned &n) {
        const size_t wk = first + it * step;
        g = (int)(wk % dst_groups);
        const size_t pc = wk / dst_groups;
        const unsigned c = (unsigned)(pc % chunks_per_blk);
        p = (int)(pc / chunks_per_blk);
        off = (size_t)c * SHMEMG_TMA_TILE;
        n = (unsigned)(nbytes - off < SHMEMG_TMA_TILE ? nbytes - off : SHMEMG_TMA_TILE);
    };
    auto issue_load = [&](size_t it) {
        int p, g; size_t off; unsigned n;
        decode(it, p, g, off, n);
        const int st = (int)(it % SHMEMG_TMA_STAGES);
        mbar_arrive_expect_tx(&full[st], n);
        bulk_g2s(stage + (size_t)st * SHMEMG_TMA_TILE, base + (size_t)p * stride + src_off + off, n, &full[st]);
    };
    for (size_t it = 0; it < mine && it < SHMEMG_TMA_STAGES - 1; ++it) issue_load(it);
    for (size_t it = 0; it < mine; ++it) {
        const int st = (int)(it % SHMEMG_TMA_STAGES);
        mbar_wait(&full[st], (unsigned)((it / SHMEMG_TMA_STAGES) & 1));
        int p, g; size_t off; unsigned n;
        decode(it, p, g, off, n);
        const int j0 = g * per_group, j1 = min(npes, j0 + per_group);
        for (int j = j0; j < j1; ++j)
            bulk_s2g(base + (size_t)j * stride + dst_off + (size_t)p * nbytes + off, stage + (size_t)st * SHMEMG_TMA_TILE, n);
        bulk_commit();
        if (it + SHMEMG_TMA_STAGES - 1 < mine) {
            bulk_wait_read<1>();
            issue_load(it + SHMEMG_TMA_STAGES - 1);
        }
    }
    bulk_wait<0>();
}
// generic byte path (unaligned sizes/offsets): plain per-(p, j) cooperative copies
__global__ void __launch_bounds__(SHMEMG_THREADS, 4)
k_fcollect_bytes(uint8_t *base, size_t stride, uint64_t dst_off, uint64_t src_off, size_t nbytes, int npes) {
    const size_t nwork = (size_t)npes * npes;
    for (size_t wk = blockIdx.x; wk < nwork; wk += gridDim.x) {
        const int j = (int)(wk % npes), p = (int)(wk / npes);
        copy_coop<4>(base + (size_t)j * stride + dst_off + (size_t)p * nbytes, base + (size_t)p * stride + src_off, nbytes,
                     threadIdx.x, SHMEMG_THREADS);
    }
}

// ---- sum_reduce, bulk-copy pipeline (offsets, stride 16-byte aligned) ---------------------------------------------------
// Work item = one column tile of RT bytes across all N windows.  Warp-specialised, one CTA per SM:
//   loader  (warp 0, lane 0) streams the tile of PE 0, 1, ... N-1 into a ring of RS stages (RG PEs per stage, one
//                            mbarrier transaction per stage), RS*RG*RT = 128 KiB in flight per SM, no registers;
//   reducers (8 warps)       thread t owns the 16 bytes at offset 16t of the tile: it adds the stages in ascending PE
//                            order (fp64 accumulators for fp32, reading 13), then writes the rounded result into one of
//                            two shared output tiles;
//   storer  (warp 1)         lane l bulk-stores the output tile to the windows l, l+32, ...; the tile is reused when its
//                            stores have finished reading it, so the next item's reduction overlaps the N-way store.
#ifndef RV
#define RV 1                                  // 16-byte vectors per reducer thread and tile
#endif
#ifndef RG
#define RG 4
#endif
#ifndef RS
#define RS 8
#endif
#define RED_THREADS 256
#define RT (RED_THREADS * 16u * RV)            // tile bytes per PE
#define RED_CTA (64 + RED_THREADS)
#define RED_SMEM ((size_t)RS * RG * RT + 2 * RT)

// ---- element math of the reductions (a15 + NEXT-2): one 16-byte vector = 4 x fp32 / 4 x int32 / 2 x fp64 / 2 x int64.
// fp32 SUM / PROD accumulate in fp64 and round once (reading 13); everything else is computed in its own type.
// Accumulators start at the operation's identity, which gives the same bits as folding the PEs in ascending order for
// NaN-free inputs (SUM starts from +0.0, so an all -0.0 column sums to +0.0: DESIGN.md reading 13).
template <int OP> __device__ __forceinline__ double red_f64(double a, double b) {
    return OP == SHMEMG_RED_SUM ? a + b : OP == SHMEMG_RED_PROD ? a * b : OP == SHMEMG_RED_MIN ? (b < a ? b : a) : (b > a ? b : a);
}
template <int OP, typename U, typename S> __device__ __forceinline__ U red_int(U a, U b) {
    switch (OP) {
    case SHMEMG_RED_SUM: return a + b;
    case SHMEMG_RED_PROD: return a * b;
    case SHMEMG_RED_MIN: return (S)b < (S)a ? b : a;
    case SHMEMG_RED_MAX: return (S)b > (S)a ? b : a;
    case SHMEMG_RED_AND: return a & b;
    case SHMEMG_RED_OR: return a | b;
    default: return a ^ b;
    }
}
template <int OP> __device__ __forceinline__ double ident_f64() {
    return OP == SHMEMG_RED_SUM ? 0.0 : OP == SHMEMG_RED_PROD ? 1.0 : OP == SHMEMG_RED_MIN ? __longlong_as_double(0x7ff0000000000000ll)
                                                                                         : __longlong_as_double(0xfff0000000000000ll);
}
template <int OP, typename U> __device__ __forceinline__ U ident_int() {
    switch (OP) {
    case SHMEMG_RED_PROD: return (U)1;
    case SHMEMG_RED_MIN: return (U)(~(U)0 >> 1);                 // signed maximum
    case SHMEMG_RED_MAX: return (U)((U)1 << (sizeof(U) * 8 - 1));  // signed minimum
    case SHMEMG_RED_AND: return (U)~(U)0;
    default: return (U)0;
    }
}
// accumulator of one 16-byte vector
template <int DT, int OP> struct RedAcc {
    double d[4];                       // F32 (4 lanes, fp64 for SUM/PROD; exact for MIN/MAX too) / F64 (2 lanes)
    unsigned long long u[2];           // I64
    unsigned w[4];                     // I32
    __device__ __forceinline__ void init() {
        if (DT == SHMEMG_F32 || DT == SHMEMG_F64) { d[0] = d[1] = d[2] = d[3] = ident_f64<OP>(); }
        else if (DT == SHMEMG_I64) { u[0] = u[1] = ident_int<OP, unsigned long long>(); }
        else { w[0] = w[1] = w[2] = w[3] = ident_int<OP, unsigned>(); }
    }
    __device__ __forceinline__ void add(const int4 &x) {
        if (DT == SHMEMG_F32) {            // fp32 -> fp64 is exact, so MIN / MAX in fp64 are exact as well
            d[0] = red_f64<OP>(d[0], (double)__int_as_float(x.x)); d[1] = red_f64<OP>(d[1], (double)__int_as_float(x.y));
            d[2] = red_f64<OP>(d[2], (double)__int_as_float(x.z)); d[3] = red_f64<OP>(d[3], (double)__int_as_float(x.w));
        } else if (DT == SHMEMG_F64) {
            d[0] = red_f64<OP>(d[0], __hiloint2double(x.y, x.x)); d[1] = red_f64<OP>(d[1], __hiloint2double(x.w, x.z));
        } else if (DT == SHMEMG_I64) {
            u[0] = red_int<OP, unsigned long long, long long>(u[0], ((unsigned long long)(unsigned)x.y << 32) | (unsigned)x.x);
            u[1] = red_int<OP, unsigned long long, long long>(u[1], ((unsigned long long)(unsigned)x.w << 32) | (unsigned)x.z);
        } else {
            w[0] = red_int<OP, unsigned, int>(w[0], (unsigned)x.x); w[1] = red_int<OP, unsigned, int>(w[1], (unsigned)x.y);
            w[2] = red_int<OP, unsigned, int>(w[2], (unsigned)x.z); w[3] = red_int<OP, unsigned, int>(w[3], (unsigned)x.w);
        }
    }
    __device__ __forceinline__ int4 result() const {
        int4 r;
        if (DT == SHMEMG_F32) {
            r.x = __float_as_int(__double2float_rn(d[0])); r.y = __float_as_int(__double2float_rn(d[1]));
            r.z = __float_as_int(__double2float_rn(d[2])); r.w = __float_as_int(__double2float_rn(d[3]));
        } else if (DT == SHMEMG_F64) {
            r.x = __double2loint(d[0]); r.y = __double2hiint(d[0]); r.z = __double2loint(d[1]); r.w = __double2hiint(d[1]);
        } else if (DT == SHMEMG_I64) {
            r.x = (int)(unsigned)u[0]; r.y = (int)(unsigned)(u[0] >> 32); r.z = (int)(unsigned)u[1]; r.w = (int)(unsigned)(u[1] >> 32);
        } else {
            r.x = (int)w[0]; r.y = (int)w[1]; r.z = (int)w[2]; r.w = (int)w[3];
        }
        return r;
    }
};

template <int DT, int OP>
__global__ void __launch_bounds__(RED_CTA, 1)
k_sum_reduce_tma(uint8_t *base, size_t stride, uint64_t dst_off, uint64_t src_off, size_t nbytes, int npes) {
    extern __shared__ __align__(1024) uint8_t smem[];
    __shared__ uint64_t full[RS], empty[RS], out_full[2], out_empty[2];
    uint8_t *out = smem + (size_t)RS * RG * RT;
    const int tid = threadIdx.x;
    const size_t ntiles = (nbytes + RT - 1) / RT;
    const int ngroups = (npes + RG - 1) / RG;
    if (tid == 0) {
        for (int s = 0; s < RS; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], RED_THREADS / 32); }
        for (int b = 0; b < 2; ++b) { mbar_init(&out_full[b], RED_THREADS / 32); mbar_init(&out_empty[b], 1); }
        mbar_init_fence();
    }
    __syncthreads();
    if (tid == 0) {
        // ---- loader ----
        unsigned it = 0;
        for (size_t c = blockIdx.x; c < ntiles; c += gridDim.x) {
            const size_t off = c * RT;
            const unsigned tb = (unsigned)(nbytes - off < RT ? nbytes - off : RT);
            const uint8_t *s0 = base + src_off + off;
            for (int g = 0; g < ngroups; ++g, ++it) {
                const unsigned s = it % RS;
                mbar_wait(&empty[s], ((it / RS) & 1u) ^ 1u);
                const int p0 = g * RG, cnt = min(RG, npes - p0);
                mbar_arrive_expect_tx(&full[s], tb * cnt);
                for (int j = 0; j < cnt; ++j)
                    bulk_g2s(smem + ((size_t)s * RG + j) * RT, s0 + (size_t)(p0 + j) * stride, tb, &full[s]);
            }
        }
    } else if (tid >= 32 && tid < 64) {
        // ---- storer ----
        const int lane = tid - 32;
        unsigned k = 0;
        for (size_t c = blockIdx.x; c < ntiles; c += gridDim.x, ++k) {
            const unsigned b = k & 1u;
            const size_t off = c * RT;
            const unsigned tb = (unsigned)(nbytes - off < RT ? nbytes - off : RT);
            mbar_wait(&out_full[b], (k >> 1) & 1u);
            for (int p = lane; p < npes; p += 32) bulk_s2g(base + (size_t)p * stride + dst_off + off, out + (size_t)b * RT, tb);
            bulk_commit();
            if (k >= 1) {                       // the previous item's stores (other tile) have read their tile
                bulk_wait_read<1>();
                __syncwarp();
                if (lane == 0) mbar_arrive(&out_empty[b ^ 1u]);
            }
        }
        bulk_wait<0>();
    } else if (tid >= 64) {
        // ---- reducers ----
        const int t = tid - 64, lane = t & 31;
        unsigned it = 0, k = 0;
        for (size_t c = blockIdx.x; c < ntiles; c += gridDim.x, ++k) {
            const size_t off = c * RT;
            const unsigned tb = (unsigned)(nbytes - off < RT ? nbytes - off : RT);
            RedAcc<DT, OP> acc[RV];
#pragma unroll
            for (int v = 0; v < RV; ++v) acc[v].init();
            for (int g = 0; g < ngroups; ++g, ++it) {
                const unsigned s = it % RS;
                mbar_wait(&full[s], (it / RS) & 1u);
                const int cnt = min(RG, npes - g * RG);
#pragma unroll
                for (int j = 0; j < RG; ++j) {
                    if (j < cnt) {
#pragma unroll
                        for (int v = 0; v < RV; ++v) {
                            const unsigned o = ((unsigned)v * RED_THREADS + (unsigned)t) * 16u;
                            if (o < tb) {
                                // ascending PE order (reading 13)
                                acc[v].add(*reinterpret_cast<const int4 *>(smem + ((size_t)s * RG + j) * RT + o));
                            }
                        }
                    }
                }
                __syncwarp();
                if (lane == 0) mbar_arrive(&empty[s]);
            }
            const unsigned b = k & 1u;
            if (k >= 2) mbar_wait(&out_empty[b], ((k >> 1) - 1u) & 1u);
#pragma unroll
            for (int v = 0; v < RV; ++v) {
                const unsigned o = ((unsigned)v * RED_THREADS + (unsigned)t) * 16u;
                if (o < tb) {
                    *reinterpret_cast<int4 *>(out + (size_t)b * RT + o) = acc[v].result();
                }
            }
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");    // generic writes -> visible to the bulk store
            __syncwarp();
            if (lane == 0) mbar_arrive(&out_full[b]);
        }
    }
}
// scalar tails / unaligned buffers: one element per thread, the same element math on one lane of a vector
template <int DT, int OP>
__global__ void k_reduce_scalar(uint8_t *base, size_t stride, uint64_t dst_off, uint64_t src_off, size_t first, size_t n,
                                int npes) {
    constexpr size_t ES = (DT == SHMEMG_F32 || DT == SHMEMG_I32) ? 4 : 8;
    for (size_t k = first + (size_t)blockIdx.x * blockDim.x + threadIdx.x; k < n; k += (size_t)gridDim.x * blockDim.x) {
        RedAcc<DT, OP> acc;
        acc.init();
        for (int p = 0; p < npes; ++p) {
            const uint8_t *q = base + (size_t)p * stride + src_off + k * ES;
            int4 x = make_int4(0, 0, 0, 0);
            x.x = (int)*reinterpret_cast<const volatile unsigned *>(q);
            if (ES == 8) x.y = (int)*reinterpret_cast<const volatile unsigned *>(q + 4);
            acc.add(x);
        }
        const int4 r = acc.result();
        for (int j = 0; j < npes; ++j) {
            uint8_t *q = base + (size_t)j * stride + dst_off + k * ES;
            *reinterpret_cast<unsigned *>(q) = (unsigned)r.x;
            if (ES == 8) *reinterpret_cast<unsigned *>(q + 4) = (unsigned)r.y;
        }
    }
}

// ---- barriers ---------------------------------------------------------------------------------------------------------
__global__ void k_barrier_epoch(CtlRegion *ctl) { atomicAdd(&ctl->barrier_epoch, 1ull); }

// One CTA per PE agent, all co-resident (cooperative launch).  Monotonic-counter barrier at GPU scope: ONE 64-bit arrival counter
// that is never reset.  An agent arrives with a fire-and-forget release `red` and polls the counter itself (relaxed loads, no L1
// invalidate per probe, one fence at the end) until it has reached the end of the round: no atomic return value to wait for, no
// last arriver, no second word -- what every poller observes IS the last arrival.  1.17 us per barrier for 128 agents.
// The first round's end is found from the counter alone (before its own arrival to barrier k an agent can only read a value in
// [k*npes, (k+1)*npes), whatever the others have done); later rounds add npes.
// Measured and not kept: the sense-reversing counter + generation word of round 1 (1.83 us: arrival atomic round
// trip + release store + poll round trip), a two-level counter tree (2.4 us: two atomic round trips in series) and a flag
// barrier without read-modify-write (every agent publishes its slot and polls all slots with 16-byte loads: 0.8 us for 8
// agents, but 1.65 - 3.15 us for 128 depending on where the agents land: 128 pollers on four L2 lines).
__device__ __forceinline__ void pe_barrier(CtlRegion *ctl, unsigned long long target) {
    // thread 0 of the CTA acts for the PE
    red_release_add_u64(&ctl->bar_arrivals, 1ull);
    while (ld_relaxed_u64(&ctl->bar_arrivals) < target) { }
    fence_acquire();
}

__global__ void __launch_bounds__(32) k_barrier_repeat(CtlRegion *ctl, uint8_t *base, size_t stride, unsigned npes,
                                                       unsigned count, unsigned long long stamp_off, int do_stamp) {
    if (threadIdx.x != 0) return;
    const unsigned p = blockIdx.x;
    const unsigned long long c0 = ld_relaxed_u64(&ctl->bar_arrivals);      // before this agent's first arrival
    unsigned long long target = c0 - c0 % npes;                              // arrivals at the start of the first round
    if (!do_stamp) {
        for (unsigned r = 0; r < count; ++r) pe_barrier(ctl, target += npes);
        return;
    }
    volatile unsigned long long *mine = reinterpret_cast<volatile unsigned long long *>(base + (size_t)p * stride + stamp_off);
    volatile unsigned long long *right =
        reinterpret_cast<volatile unsigned long long *>(base + (size_t)((p + 1) % npes) * stride + stamp_off);
    unsigned long long bad = 0;
    for (unsigned r = 1; r <= count; ++r) {
        right[r & 1] = r;                 // "put" r into slot r&1 of the right neighbour
        pe_barrier(ctl, target += npes);  // barrier_all: the put is complete and visible
        if (mine[r & 1] != r) bad++;      // my left neighbour's stamp of THIS round must be there
        // no second barrier needed: slot r&1 is next written in round r+2, i.e. after barrier r+1, which this
        // agent only reaches after the read above
    }
    mine[2] += bad;
}

// Recovery after a kernel that did not finish its rounds (aborted, timed out, or a user kernel in which fewer than npes agents
// reached a barrier): the monotonic arrival counters find their round from the count alone, so a residue would make every later
// barrier of the world release early.  Rounds the counters up to the next round boundary and clears the last-arriver counters.
__global__ void k_realign_counters(CtlRegion *ctl, unsigned npes) {
    const unsigned t = threadIdx.x;
    if (t == 0) {
        const unsigned long long c = ctl->bar_arrivals, r = c % npes;
        if (r) ctl->bar_arrivals = c + (npes - r);
        const unsigned h = ctl->hot_done, hr = h % 16u;                  // 16 sampling CTAs per call (2^32 is a multiple of 16)
        if (hr) ctl->hot_done = h + (16u - hr);
        ctl->amo_done = 0;
    }
    for (unsigned i = t; i < SHMEMG_SIG_SLOTS; i += blockDim.x) ctl->sig_counter[i] = 0;
}

extern "C" int shmemg_realign_counters_on_stream(shmemg_world_t *w, void *stream) {
    if (!w) return SHMEMG_ERR_ARG;
    k_realign_counters<<<1, 256, 0, (cudaStream_t)stream>>>(w->ctl, (unsigned)w->npes);
    SHMEMG_CUDA(w, cudaGetLastError());
    return SHMEMG_OK;
}

// ---------------------------------------------------------------------------------------------------------
// host entry points
// ---------------------------------------------------------------------------------------------------------
static int collectives_smem_attr(shmemg_world *w) {
    if (w->smem_attr_coll) return SHMEMG_OK;
    SHMEMG_CUDA(w, cudaFuncSetAttribute(k_alltoall_tma, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SHMEMG_TMA_SMEM));
    SHMEMG_CUDA(w, cudaFuncSetAttribute(k_fcollect_tma, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SHMEMG_TMA_SMEM));
    SHMEMG_CUDA(w, cudaFuncSetAttribute(k_alltoalls_tma, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SHMEMG_TMA_SMEM));
    w->smem_attr_coll = true;
    return SHMEMG_OK;
}

static bool ranges_overlap(uint64_t a, uint64_t b, uint64_t n_a, uint64_t n_b) { return a < b + n_b && b < a + n_a; }

extern "C" int shmemg_alltoall_on_stream(shmemg_world_t *w, uint64_t dest_off, uint64_t source_off, size_t nbytes,
                                         void *stream) {
    if (!w) return SHMEMG_ERR_ARG;
    const uint64_t tot = (uint64_t)nbytes * w->npes;
    if (!shmemg_in_range(w, dest_off, tot) || !shmemg_in_range(w, source_off, tot)) return SHMEMG_ERR_RANGE;
    if (nbytes == 0) return SHMEMG_OK;
    if (ranges_overlap(dest_off, source_off, tot, tot)) return SHMEMG_ERR_OVERLAP;
    cudaStream_t st = (cudaStream_t)stream;
    if (((dest_off | source_off | nbytes | w->stride) & 15) == 0 && !w->tile_bytes_override) {
        int rc = collectives_smem_attr(w);
        if (rc) return rc;
        const unsigned cpb = (unsigned)((nbytes + SHMEMG_TMA_TILE - 1) / SHMEMG_TMA_TILE);
        const uint64_t nwork = (uint64_t)w->npes * w->npes * cpb;
        const unsigned grid = (unsigned)(nwork < (uint64_t)w->sm_count ? nwork : (uint64_t)w->sm_count);
        k_alltoall_tma<<<grid, 32, SHMEMG_TMA_SMEM, st>>>(w->base, w->stride, dest_off, source_off, nbytes, w->npes, cpb);
        SHMEMG_CUDA(w, cudaGetLastError());
        return SHMEMG_OK;
    }
    const uint64_t maxgrid = (uint64_t)w->sm_count * w->ctas_per_sm;
    unsigned chunk = 65536;
    if (w->tile_bytes_override) chunk = (unsigned)w->tile_bytes_override;
    else
        while (chunk > 4096 && (uint64_t)w->npes * w->npes * ((nbytes + chunk - 1) / chunk) < maxgrid * 8) chunk >>= 1;
    const unsigned cpb = (unsigned)((nbytes + chunk - 1) / chunk);
    const uint64_t nwork = (uint64_t)w->npes * w->npes * cpb;
    const unsigned grid = (unsigned)(nwork < maxgrid ? nwork : maxgrid);
    k_alltoall<<<grid, SHMEMG_THREADS, 0, st>>>(w->base, w->stride, dest_off, source_off, nbytes, w->npes, chunk, cpb);
    SHMEMG_CUDA(w, cudaGetLastError());
    return SHMEMG_OK;
}

extern "C" int shmemg_alltoalls_on_stream(shmemg_world_t *w, uint64_t dest_off, uint64_t source_off, uint64_t dst_pe_stride,
                                          uint64_t src_pe_stride, uint64_t dst_block_stride, uint64_t src_block_stride,
                                          size_t block_bytes, size_t nblocks, void *stream) {
    if (!w) return SHMEMG_ERR_ARG;
    if (block_bytes == 0 || nblocks == 0) return SHMEMG_OK;
    const uint64_t N = (uint64_t)w->npes, hb = w->heap_bytes;
    // spans (overflow-safe: every term is checked against the heap size first)
    if (block_bytes > hb || (N > 1 && (dst_pe_stride > hb || src_pe_stride > hb)) ||
        (nblocks > 1 && (dst_block_stride > hb || src_block_stride > hb)) || nblocks > hb)
        return SHMEMG_ERR_RANGE;
    const uint64_t dspan = (N - 1) * dst_pe_stride + (nblocks - 1) * dst_block_stride + block_bytes;
    const uint64_t sspan = (N - 1) * src_pe_stride + (nblocks - 1) * src_block_stride + block_bytes;
    if (!shmemg_in_range(w, dest_off, dspan) || !shmemg_in_range(w, source_off, sspan)) return SHMEMG_ERR_RANGE;
    if (ranges_overlap(dest_off, source_off, dspan, sspan)) return SHMEMG_ERR_OVERLAP;
    // destination blocks of one PE pair / of two source PEs that cannot help overlapping
    if ((nblocks > 1 && dst_block_stride < block_bytes) || (N > 1 && dst_pe_stride < block_bytes)) return SHMEMG_ERR_OVERLAP;
    A2asArgs a{w->base, w->stride, dest_off, source_off, dst_pe_stride, src_pe_stride, dst_block_stride, src_block_stride,
               block_bytes, nblocks, w->npes};
    const uint64_t all = dest_off | source_off | dst_pe_stride | src_pe_stride | dst_block_stride | src_block_stride | block_bytes |
                         (uint64_t)w->stride | (uint64_t)(uintptr_t)w->base;
    cudaStream_t st = (cudaStream_t)stream;
    const uint64_t maxgrid = (uint64_t)w->sm_count * w->ctas_per_sm;
    if (block_bytes >= 1024 && (all & 15) == 0 && !w->tile_bytes_override) {
        int rc = collectives_smem_attr(w);
        if (rc) return rc;
        const unsigned cpb = (unsigned)((block_bytes + SHMEMG_TMA_TILE - 1) / SHMEMG_TMA_TILE);
        const uint64_t nwork = N * nblocks * N * cpb;
        k_alltoalls_tma<<<(unsigned)(nwork < (uint64_t)w->sm_count ? nwork : (uint64_t)w->sm_count), 32, SHMEMG_TMA_SMEM, st>>>(a, cpb);
    } else if ((block_bytes == 4 || block_bytes == 8 || block_bytes == 16) && (all & (block_bytes - 1)) == 0) {
        const uint64_t n = N * N * nblocks;
        const unsigned grid = (unsigned)((n + 255) / 256 < maxgrid * 2 ? (n + 255) / 256 : maxgrid * 2);
        if (block_bytes == 4) k_alltoalls_elem<unsigned><<<grid, 256, 0, st>>>(a);
        else if (block_bytes == 8) k_alltoalls_elem<unsigned long long><<<grid, 256, 0, st>>>(a);
        else k_alltoalls_elem<int4><<<grid, 256, 0, st>>>(a);
    } else {
        const unsigned cpb = (unsigned)((block_bytes + 16383) / 16384);
        const uint64_t nwork = N * nblocks * N * cpb;
        k_alltoalls_generic<<<(unsigned)(nwork < maxgrid ? nwork : maxgrid), SHMEMG_THREADS, 0, st>>>(a, cpb);
    }
    SHMEMG_CUDA(w, cudaGetLastError());
    return SHMEMG_OK;
}

extern "C" int shmemg_fcollect_on_stream(shmemg_world_t *w, uint64_t dest_off, uint64_t source_off, size_t nbytes,
                                         void *stream) {
    if (!w) return SHMEMG_ERR_ARG;
    const uint64_t tot = (uint64_t)nbytes * w->npes;
    if (!shmemg_in_range(w, dest_off, tot) || !shmemg_in_range(w, source_off, nbytes)) return SHMEMG_ERR_RANGE;
    if (nbytes == 0) return SHMEMG_OK;
    if (ranges_overlap(dest_off, source_off, tot, nbytes)) return SHMEMG_ERR_OVERLAP;
    const uint64_t maxgrid = (uint64_t)w->sm_count * w->ctas_per_sm;
    cudaStream_t st = (cudaStream_t)stream;
    if (((dest_off | source_off | nbytes | w->stride) & 15) == 0 && !w->tile_bytes_override) {
        int rc = collectives_smem_attr(w);
        if (rc) return rc;
        const unsigned cpb = (unsigned)((nbytes + SHMEMG_TMA_TILE - 1) / SHMEMG_TMA_TILE);
        // One destination per work item: consecutive items (one per CTA) store the same source chunk, which is read from
        // HBM once and from L2 by the others.  Measured on C5 (profiles/r01c): 93.0 us against 96.9 us with 8
        // destinations per loaded tile; the write-only ceiling of bulk stores on this box is 88 us.
        int groups = w->npes;
#ifdef SHMEMG_EXPERIMENTS
        if (const char *e = getenv("SHMEMG_FCOLLECT_GROUPS")) {
            groups = atoi(e);
            if (groups < 1 || groups > w->npes) groups = w->npes;
        }
#endif
        const uint64_t nwork = (uint64_t)w->npes * cpb * groups;
        const unsigned grid = (unsigned)(nwork < (uint64_t)w->sm_count ? nwork : (uint64_t)w->sm_count);
        k_fcollect_tma<<<grid, 32, SHMEMG_TMA_SMEM, st>>>(w->base, w->stride, dest_off, source_off, nbytes, w->npes, cpb, groups);
    } else if (((dest_off | source_off | nbytes | w->stride) & 15) == 0) {
        constexpr int VPT = 4;                                  // 256 threads * 4 * 16 B = 16 KiB per work item
        const unsigned cpb = (unsigned)(((nbytes >> 4) + SHMEMG_THREADS * VPT - 1) / (SHMEMG_THREADS * VPT));
        int groups = 1;                                         // split destinations until the grid is full
        while (groups < w->npes && (uint64_t)w->npes * cpb * groups < maxgrid * 4) groups <<= 1;
        if (groups > w->npes) groups = w->npes;
        const uint64_t nwork = (uint64_t)w->npes * cpb * groups;
        const unsigned grid = (unsigned)(nwork < maxgrid ? nwork : maxgrid);
        k_fcollect_vec<VPT><<<grid, SHMEMG_THREADS, 0, st>>>(w->base, w->stride, dest_off, source_off, nbytes, w->npes,
                                                             cpb, groups);
    } else {
        const uint64_t nwork = (uint64_t)w->npes * w->npes;
        const unsigned grid = (unsigned)(nwork < maxgrid ? nwork : maxgrid);
        k_fcollect_bytes<<<grid, SHMEMG_THREADS, 0, st>>>(w->base, w->stride, dest_off, source_off, nbytes, w->npes);
    }
    SHMEMG_CUDA(w, cudaGetLastError());
    return SHMEMG_OK;
}

template <int DT, int OP>
static void launch_reduce(shmemg_world *w, uint64_t dest_off, uint64_t source_off, size_t nvec, size_t first, size_t nreduce,
                          cudaStream_t st) {
    if (nvec) {
        if (!w->smem_attr_red[DT][OP]) {
            if (cudaFuncSetAttribute(k_sum_reduce_tma<DT, OP>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)RED_SMEM) != cudaSuccess)
                return;                                    // the caller's cudaGetLastError reports it
            w->smem_attr_red[DT][OP] = true;
        }
        const size_t nb = nvec << 4, ntiles = (nb + RT - 1) / RT;
        const unsigned grid = (unsigned)(ntiles < (size_t)w->sm_count ? ntiles : (size_t)w->sm_count);
        k_sum_reduce_tma<DT, OP><<<grid, RED_CTA, RED_SMEM, st>>>(w->base, w->stride, dest_off, source_off, nb, w->npes);
    }
    if (first < nreduce) {
        size_t blocks = (nreduce - first + 255) / 256;
        if (blocks > 4096) blocks = 4096;
        k_reduce_scalar<DT, OP><<<(unsigned)blocks, 256, 0, st>>>(w->base, w->stride, dest_off, source_off, first, nreduce, w->npes);
    }
}
template <int DT>
static int launch_reduce_op(shmemg_world *w, int op, uint64_t d, uint64_t s, size_t nvec, size_t first, size_t n, cudaStream_t st) {
    switch (op) {
    case SHMEMG_RED_SUM: launch_reduce<DT, SHMEMG_RED_SUM>(w, d, s, nvec, first, n, st); break;
    case SHMEMG_RED_PROD: launch_reduce<DT, SHMEMG_RED_PROD>(w, d, s, nvec, first, n, st); break;
    case SHMEMG_RED_MIN: launch_reduce<DT, SHMEMG_RED_MIN>(w, d, s, nvec, first, n, st); break;
    case SHMEMG_RED_MAX: launch_reduce<DT, SHMEMG_RED_MAX>(w, d, s, nvec, first, n, st); break;
    default:
        if (DT == SHMEMG_F32 || DT == SHMEMG_F64) return SHMEMG_ERR_ARG;       // no bitwise reductions on floating point
        if (op == SHMEMG_RED_AND) launch_reduce<DT == SHMEMG_F32 || DT == SHMEMG_F64 ? SHMEMG_I64 : DT, SHMEMG_RED_AND>(w, d, s, nvec, first, n, st);
        else if (op == SHMEMG_RED_OR) launch_reduce<DT == SHMEMG_F32 || DT == SHMEMG_F64 ? SHMEMG_I64 : DT, SHMEMG_RED_OR>(w, d, s, nvec, first, n, st);
        else launch_reduce<DT == SHMEMG_F32 || DT == SHMEMG_F64 ? SHMEMG_I64 : DT, SHMEMG_RED_XOR>(w, d, s, nvec, first, n, st);
    }
    return SHMEMG_OK;
}

extern "C" int shmemg_reduce_on_stream(shmemg_world_t *w, int op, int dtype, uint64_t dest_off, uint64_t source_off,
                                       size_t nreduce, void *stream) {
    if (!w || dtype < SHMEMG_F32 || dtype > SHMEMG_F64 || op < SHMEMG_RED_SUM || op > SHMEMG_RED_XOR) return SHMEMG_ERR_ARG;
    if ((dtype == SHMEMG_F32 || dtype == SHMEMG_F64) && op >= SHMEMG_RED_AND) return SHMEMG_ERR_ARG;
    const size_t esz = (dtype == SHMEMG_F32 || dtype == SHMEMG_I32) ? 4 : 8;
    const uint64_t tot = (uint64_t)nreduce * esz;
    if (!shmemg_in_range(w, dest_off, tot) || !shmemg_in_range(w, source_off, tot)) return SHMEMG_ERR_RANGE;
    if ((dest_off | source_off) & (esz - 1)) return SHMEMG_ERR_ALIGN;
    if (dest_off != source_off && ranges_overlap(dest_off, source_off, tot, tot)) return SHMEMG_ERR_OVERLAP;
    if (nreduce == 0) return SHMEMG_OK;
    cudaStream_t st = (cudaStream_t)stream;
    const bool vec_ok = ((dest_off | source_off | w->stride) & 15) == 0;
    const size_t nvec = vec_ok ? tot >> 4 : 0;
    const size_t first = nvec * (16 / esz);
    int rc;
    switch (dtype) {
    case SHMEMG_F32: rc = launch_reduce_op<SHMEMG_F32>(w, op, dest_off, source_off, nvec, first, nreduce, st); break;
    case SHMEMG_I64: rc = launch_reduce_op<SHMEMG_I64>(w, op, dest_off, source_off, nvec, first, nreduce, st); break;
    case SHMEMG_I32: rc = launch_reduce_op<SHMEMG_I32>(w, op, dest_off, source_off, nvec, first, nreduce, st); break;
    default: rc = launch_reduce_op<SHMEMG_F64>(w, op, dest_off, source_off, nvec, first, nreduce, st); break;
    }
    if (rc) return rc;
    SHMEMG_CUDA(w, cudaGetLastError());
    return SHMEMG_OK;
}

extern "C" int shmemg_sum_reduce_on_stream(shmemg_world_t *w, int dtype, uint64_t dest_off, uint64_t source_off,
                                           size_t nreduce, void *stream) {
    if (dtype != SHMEMG_F32 && dtype != SHMEMG_I64) return SHMEMG_ERR_ARG;
    return shmemg_reduce_on_stream(w, SHMEMG_RED_SUM, dtype, dest_off, source_off, nreduce, stream);
}

extern "C" int shmemg_barrier_all_on_stream(shmemg_world_t *w, void *stream) {
    if (!w) return SHMEMG_ERR_ARG;
    k_barrier_epoch<<<1, 1, 0, (cudaStream_t)stream>>>(w->ctl);
    SHMEMG_CUDA(w, cudaGetLastError());
    return SHMEMG_OK;
}

extern "C" int shmemg_barrier_all_repeat_on_stream(shmemg_world_t *w, uint32_t count, uint64_t stamp_off, void *stream) {
    if (!w) return SHMEMG_ERR_ARG;
    const int do_stamp = stamp_off != UINT64_MAX;
    if (do_stamp) {
        if (!shmemg_in_range(w, stamp_off, 24)) return SHMEMG_ERR_RANGE;
        if (stamp_off & 7) return SHMEMG_ERR_ALIGN;
    }
    if (count == 0) return SHMEMG_OK;
    int per_sm = 0;
    SHMEMG_CUDA(w, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_barrier_repeat, 32, 0));
    if ((long long)per_sm * w->sm_count < w->npes) return SHMEMG_ERR_NOMEM;   // agents could not all be co-resident
    CtlRegion *ctl = w->ctl;
    uint8_t *base = w->base;
    size_t stride = w->stride;
    unsigned npes = (unsigned)w->npes;
    unsigned long long so = do_stamp ? stamp_off : 0;
    int ds = do_stamp;
    void *args[] = {&ctl, &base, &stride, &npes, &count, &so, &ds};
    SHMEMG_CUDA(w, cudaLaunchCooperativeKernel((void *)k_barrier_repeat, dim3(npes), dim3(32), args, 0, (cudaStream_t)stream));
    return SHMEMG_OK;
}

extern "C" uint64_t shmemg_barrier_epoch(shmemg_world_t *w, void *stream) {
    if (!w) return 0;
    unsigned long long v = 0;
    if (cudaMemcpyAsync(&v, &w->ctl->barrier_epoch, 8, cudaMemcpyDeviceToHost, (cudaStream_t)stream) != cudaSuccess) return 0;
    cudaStreamSynchronize((cudaStream_t)stream);
    return v;
}
