// shard.cu -- PE -> GPU sharding over a load-store fabric.
//
// One world per GPU (one process per GPU in the usual deployment); G = nshards worlds form one global OpenSHMEM world.
// Placement: GLOBAL PE g lives on shard g mod G as that shard's LOCAL PE g div G (reading 42).  Every shard maps the
// slabs of the others (CUDA IPC between processes, plain peer pointers inside one process), so
//     address(g, off) = peer_base[g mod G] + (g div G) * stride + off
// is an ordinary global-memory address on THIS device and every operation is a kernel of the initiating shard that loads
// from / stores to / performs atomics on peer memory over NVLink 5 / NVSwitch:
//   put / get / put_signal   register-path copy (16-byte vector accesses where the alignment allows), last-arriver signal;
//   AMO batches              red / atom at SYSTEM scope (the atomicity domain is the fabric, not one GPU's L2);
//   alltoall                 every (local source PE, global destination PE) block is pushed into the destination's window
//                            (bulk copies through shared memory when everything is 16-byte aligned);
//   barrier                  one kernel per shard: arrive on EVERY shard's counter (red.release.sys), wait for the own one.
// Nothing here touches the single-GPU kernels; with nshards == 1 the g-calls compute what their unsharded counterparts compute.
#include <stddef.h>
#include <string.h>

#include "tma_stream.cuh"

struct ShardView {                      // by value into the kernels
    uint8_t *base[SHMEMG_MAX_SHARDS];
    unsigned long long stride;
    int nshards, shard, npes_local;
};

__device__ __forceinline__ uint8_t *g_addr(const ShardView &v, int gpe, unsigned long long off) {
    return v.base[gpe % v.nshards] + (unsigned long long)(gpe / v.nshards) * v.stride + off;
}

// ---- memory-model primitives at SYSTEM scope --------------------------------------------------------------------------
__device__ __forceinline__ void fence_sys() { asm volatile("fence.acq_rel.sys;" ::: "memory"); }
__device__ __forceinline__ void red_release_sys_add_u64(unsigned long long *p, unsigned long long v) {
    asm volatile("red.release.sys.global.add.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}
__device__ __forceinline__ void exch_release_sys_u64(unsigned long long *p, unsigned long long v) {
    asm volatile("{ .reg .b64 t; atom.release.sys.global.exch.b64 t, [%0], %1; }" ::"l"(p), "l"(v) : "memory");
}
__device__ __forceinline__ unsigned long long ld_relaxed_sys_u64(const unsigned long long *p) {
    unsigned long long v;
    asm volatile("ld.relaxed.sys.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}

// ---- put / get / put_signal: grid-stride over tiles, optional last-arriver signal at system scope -----------------------
__global__ void __launch_bounds__(SHMEMG_THREADS, 4)
k_shard_copy(uint8_t *dst, const uint8_t *src, size_t nbytes, unsigned tile_bytes, unsigned long long *sig,
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
            fence_sys();                                   // this CTA's stores, possibly to peer memory
            if (atomicAdd(counter, 1u) == gridDim.x - 1) { // the counter is local: GPU scope
                fence_sys();
                *counter = 0;
                if (sig_op == SHMEMG_SIGNAL_ADD) red_release_sys_add_u64(sig, sig_value);
                else exch_release_sys_u64(sig, sig_value);
            }
        }
    }
}

__global__ void k_shard_wait_until(const unsigned long long *sig, int cmp, unsigned long long value) {
    while (!cmp_u64(cmp, ld_relaxed_sys_u64(sig), value)) __nanosleep(100);
    fence_sys();
}

// ---- AMO batches with global targets: system-scope L2 / fabric atomics --------------------------------------------------
struct ShardAmoArgs {
    ShardView v;
    unsigned long long sym_off;
    const int *tgt;
    const void *idx;
    const unsigned long long *val, *cond;
    unsigned long long val_s, cond_s;
    unsigned long long *fetched;
    size_t n;
};
template <int IDXB> struct SIdxT;
template <> struct SIdxT<4> { typedef unsigned int type; };
template <> struct SIdxT<8> { typedef unsigned long long type; };

template <int IDXB, int OP>
__global__ void __launch_bounds__(256) k_shard_amo(const ShardAmoArgs a) {
    typedef typename SIdxT<IDXB>::type idx_t;
    const idx_t *__restrict__ idx = reinterpret_cast<const idx_t *>(a.idx);
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < a.n; i += (size_t)gridDim.x * blockDim.x) {
        unsigned long long *word = reinterpret_cast<unsigned long long *>(g_addr(a.v, a.tgt[i], a.sym_off) + 8ull * (unsigned long long)idx[i]);
        const unsigned long long v = a.val ? a.val[i] : a.val_s;
        if (OP == SHMEMG_OP_ATOMIC_ADD) {
            asm volatile("red.relaxed.sys.global.add.u64 [%0], %1;" ::"l"(word), "l"(v) : "memory");
        } else if (OP == SHMEMG_OP_ATOMIC_FETCH_ADD) {
            unsigned long long old;
            asm volatile("atom.relaxed.sys.global.add.u64 %0, [%1], %2;" : "=l"(old) : "l"(word), "l"(v) : "memory");
            a.fetched[i] = old;
        } else {
            const unsigned long long c = a.cond ? a.cond[i] : a.cond_s;
            unsigned long long old;
            asm volatile("atom.relaxed.sys.global.cas.b64 %0, [%1], %2, %3;" : "=l"(old) : "l"(word), "l"(c), "l"(v) : "memory");
            a.fetched[i] = old;
        }
    }
}

// ---- alltoall: local PE l (global s = l*G + shard) pushes block j of its source into global PE j's window at block s ----
__global__ void __launch_bounds__(SHMEMG_THREADS, 4)
k_shard_alltoall(const ShardView v, unsigned long long dst_off, unsigned long long src_off, size_t nbytes, unsigned chunk) {
    const int gn = v.nshards * v.npes_local;
    const size_t chunks = (nbytes + chunk - 1) / chunk;
    const size_t items = (size_t)v.npes_local * gn * chunks;
    for (size_t it = blockIdx.x; it < items; it += gridDim.x) {
        const size_t c = it % chunks;
        const int j = (int)((it / chunks) % gn);                       // destination (global)
        const int l = (int)(it / chunks / gn);                          // source (local)
        const int s = l * v.nshards + v.shard;                          // source (global)
        const size_t off = c * chunk;
        const size_t n = nbytes - off < chunk ? nbytes - off : chunk;
        const uint8_t *src = v.base[v.shard] + (unsigned long long)l * v.stride + src_off + (size_t)j * nbytes + off;
        uint8_t *dst = g_addr(v, j, dst_off) + (size_t)s * nbytes + off;
        copy_coop<8>(dst, src, n, threadIdx.x, SHMEMG_THREADS);
    }
}

// bulk-copy form (everything 16-byte aligned): one issuing thread per CTA streams (source PE, destination PE, chunk) items
// through shared memory; the bulk store's destination is the destination shard's window -- local HBM or peer memory alike
__global__ void __launch_bounds__(32)
k_shard_alltoall_tma(const ShardView v, unsigned long long dst_off, unsigned long long src_off, size_t nbytes) {
    extern __shared__ __align__(1024) uint8_t stage[];
    __shared__ uint64_t full[SHMEMG_TMA_STAGES];
    if (threadIdx.x != 0) return;
    tma_stream_init(full);
    const int gn = v.nshards * v.npes_local;
    const size_t chunks = (nbytes + SHMEMG_TMA_TILE - 1) / SHMEMG_TMA_TILE;
    const size_t items = (size_t)v.npes_local * gn * chunks;
    tma_stream_copy(stage, full, blockIdx.x, gridDim.x, items, [&](size_t it, const uint8_t *&s, uint8_t *&d, unsigned &n) {
        const size_t c = it % chunks;
        const int j = (int)((it / chunks) % gn), l = (int)(it / chunks / gn);
        const size_t off = c * SHMEMG_TMA_TILE;
        n = (unsigned)(nbytes - off < SHMEMG_TMA_TILE ? nbytes - off : SHMEMG_TMA_TILE);
        s = v.base[v.shard] + (unsigned long long)l * v.stride + src_off + (size_t)j * nbytes + off;
        d = g_addr(v, j, dst_off) + (size_t)(l * v.nshards + v.shard) * nbytes + off;
    });
}

// ---- fcollect: local PE l (global s) pushes its block into block s of every global PE's destination --------------------
__global__ void __launch_bounds__(SHMEMG_THREADS, 4)
k_shard_fcollect(const ShardView v, unsigned long long dst_off, unsigned long long src_off, size_t nbytes, unsigned chunk) {
    const int gn = v.nshards * v.npes_local;
    const size_t chunks = (nbytes + chunk - 1) / chunk;
    const size_t items = (size_t)v.npes_local * chunks * gn;
    for (size_t it = blockIdx.x; it < items; it += gridDim.x) {      // consecutive items share the source chunk (L2)
        const int j = (int)(it % gn);
        const size_t c = (it / gn) % chunks;
        const int l = (int)(it / gn / chunks);
        const int s = l * v.nshards + v.shard;
        const size_t off = c * chunk;
        const size_t n = nbytes - off < chunk ? nbytes - off : chunk;
        copy_coop<8>(g_addr(v, j, dst_off) + (size_t)s * nbytes + off, v.base[v.shard] + (unsigned long long)l * v.stride + src_off + off,
                     n, threadIdx.x, SHMEMG_THREADS);
    }
}

// ---- sum_reduce = reduce-scatter + all-gather over the fabric: this shard owns elements [e0, e1) -------------------------
// One element per thread and trip: NP peer / local loads in ascending GLOBAL PE order (fp32 accumulated in fp64, one rounding;
// int64 wraps), then NP stores.  The loads of one element by consecutive threads are coalesced per window.
template <typename T> struct GAcc;
template <> struct GAcc<float> { typedef double acc_t; };
template <> struct GAcc<long long> { typedef unsigned long long acc_t; };
template <typename T>
__global__ void __launch_bounds__(256) k_shard_sum_reduce(const ShardView v, unsigned long long dst_off, unsigned long long src_off,
                                                          size_t e0, size_t e1) {
    typedef typename GAcc<T>::acc_t acc_t;
    const int gn = v.nshards * v.npes_local;
    for (size_t e = e0 + (size_t)blockIdx.x * blockDim.x + threadIdx.x; e < e1; e += (size_t)gridDim.x * blockDim.x) {
        acc_t acc = 0;                                               // fp: +0.0 + x_0 + x_1 + ... (reading 13)
        for (int g = 0; g < gn; ++g)
            acc += (acc_t)*reinterpret_cast<const volatile T *>(g_addr(v, g, src_off) + e * sizeof(T));
        const T r = (T)acc;
        for (int g = 0; g < gn; ++g) *reinterpret_cast<T *>(g_addr(v, g, dst_off) + e * sizeof(T)) = r;
    }
}

// ---- barrier of the shards' streams ------------------------------------------------------------------------------------
// Everything this shard's stream did before the kernel is complete (kernel boundary); the system-scope release makes it visible to
// whoever observes the arrival.  Each shard's counter advances by G per barrier; epoch = barriers enqueued so far on this world.
__global__ void k_shard_barrier(const ShardView v, unsigned long long ctl_off, unsigned long long bar_off, unsigned long long epoch) {
    if (threadIdx.x != 0 || blockIdx.x != 0) return;
    fence_sys();
    for (int s = 0; s < v.nshards; ++s)
        red_release_sys_add_u64(reinterpret_cast<unsigned long long *>(v.base[s] + ctl_off + bar_off), 1ull);
    const unsigned long long *mine = reinterpret_cast<const unsigned long long *>(v.base[v.shard] + ctl_off + bar_off);
    while (ld_relaxed_sys_u64(mine) < epoch * (unsigned long long)v.nshards) __nanosleep(100);
    fence_sys();
}

// ---------------------------------------------------------------------------------------------------------------------------
// host
// ---------------------------------------------------------------------------------------------------------------------------
extern "C" int shmemg_shard_of(int gpe, int nshards) { return (gpe < 0 || nshards < 1) ? SHMEMG_ERR_ARG : gpe % nshards; }
extern "C" int shmemg_shard_local_index(int gpe, int nshards) { return (gpe < 0 || nshards < 1) ? SHMEMG_ERR_ARG : gpe / nshards; }
extern "C" int shmemg_shard_global_pe(int shard, int local_pe, int nshards) {
    return (nshards < 1 || shard < 0 || shard >= nshards || local_pe < 0) ? SHMEMG_ERR_ARG : local_pe * nshards + shard;
}

extern "C" int shmemg_shard_init(shmemg_world_t *w, int nshards, int my_shard) {
    if (!w || nshards < 1 || nshards > SHMEMG_MAX_SHARDS || my_shard < 0 || my_shard >= nshards) return SHMEMG_ERR_ARG;
    if (w->nshards) return SHMEMG_ERR_ARG;                       // once
    w->nshards = nshards;
    w->shard = my_shard;
    w->peer_base[my_shard] = w->base;
    return SHMEMG_OK;
}

extern "C" int shmemg_shard_global_npes(const shmemg_world_t *w) { return (w && w->nshards) ? w->nshards * w->npes : SHMEMG_ERR_ARG; }

// the allocation that holds the slab: cudaIpcGetMemHandle names whole allocations (the slab may sit inside a pooled block)
static int alloc_range(void *p, void **base, size_t *size) {
    typedef int (*fn_t)(unsigned long long *, size_t *, unsigned long long);
    void *fn = nullptr;
    cudaDriverEntryPointQueryResult qr;
    if (cudaGetDriverEntryPoint("cuMemGetAddressRange", &fn, cudaEnableDefault, &qr) != cudaSuccess || !fn) return SHMEMG_ERR_CUDA;
    unsigned long long b = 0;
    size_t s = 0;
    if (((fn_t)fn)(&b, &s, (unsigned long long)(uintptr_t)p) != 0) return SHMEMG_ERR_CUDA;
    *base = (void *)(uintptr_t)b;
    *size = s;
    return SHMEMG_OK;
}

extern "C" int shmemg_shard_export(shmemg_world_t *w, void *ipc_handle64_out, uint64_t *offset_out) {
    if (!w || !w->nshards || !ipc_handle64_out || !offset_out) return SHMEMG_ERR_ARG;
    static_assert(sizeof(cudaIpcMemHandle_t) == 64, "a CUDA IPC handle is 64 bytes");
    void *abase = nullptr;
    size_t asize = 0;
    int rc = alloc_range(w->base, &abase, &asize);
    if (rc) return rc;
    cudaIpcMemHandle_t h;
    SHMEMG_CUDA(w, cudaIpcGetMemHandle(&h, abase));
    memcpy(ipc_handle64_out, &h, 64);
    *offset_out = (uint64_t)((uint8_t *)w->base - (uint8_t *)abase);
    return SHMEMG_OK;
}

// A peer slab must be device memory that THIS world's GPU can load, store and -- because signals, the shard barrier and the AMO
// batches use red / atom at system scope -- atomically update.  A slab on the world's own GPU passes at once; for one on another
// GPU peer access is required (and enabled here) and the link must support native atomics (NVLink does; PCIe P2P does not).
// Without this check the first g-call to an unreachable slab is an illegal-address fault, and atomics over a link without
// native support silently lose their atomicity.
static int peer_reachable(shmemg_world *w, const void *p) {
    cudaPointerAttributes at;
    SHMEMG_CUDA(w, cudaPointerGetAttributes(&at, p));
    if (at.type != cudaMemoryTypeDevice) {
        w->last_cuda_error = "shard attach: the peer slab is not device memory";
        return SHMEMG_ERR_ARG;
    }
    if (at.device == w->device) return SHMEMG_OK;
    int cur = -1;
    SHMEMG_CUDA(w, cudaGetDevice(&cur));
    if (cur != w->device) SHMEMG_CUDA(w, cudaSetDevice(w->device));
    int rc = SHMEMG_OK, can = 0, native_atomics = 0;
    cudaError_t e = cudaDeviceCanAccessPeer(&can, w->device, at.device);
    if (e == cudaSuccess && can) {
        e = cudaDeviceEnablePeerAccess(at.device, 0);
        if (e == cudaErrorPeerAccessAlreadyEnabled) { cudaGetLastError(); e = cudaSuccess; }
    }
    if (e == cudaSuccess && can) e = cudaDeviceGetP2PAttribute(&native_atomics, cudaDevP2PAttrNativeAtomicSupported, w->device, at.device);
    if (e != cudaSuccess) rc = shmemg_cuda_fail(w, e, "shard attach: peer access");
    else if (!can || !native_atomics) {
        w->last_cuda_error = "shard attach: device " + std::to_string(w->device) + (can ? " has no native atomics on" : " cannot access") +
                             " the memory of device " + std::to_string(at.device);
        rc = SHMEMG_ERR_NODEVICE;
    }
    if (cur != w->device) cudaSetDevice(cur);
    return rc;
}

extern "C" int shmemg_shard_attach_ipc(shmemg_world_t *w, int shard, const void *ipc_handle64, uint64_t offset) {
    if (!w || !w->nshards || !ipc_handle64 || shard < 0 || shard >= w->nshards || shard == w->shard) return SHMEMG_ERR_ARG;
    if (w->peer_base[shard]) return SHMEMG_ERR_ARG;
    cudaIpcMemHandle_t h;
    memcpy(&h, ipc_handle64, 64);
    void *p = nullptr;
    SHMEMG_CUDA(w, cudaIpcOpenMemHandle(&p, h, cudaIpcMemLazyEnablePeerAccess));
    const int rc = peer_reachable(w, p);
    if (rc) { cudaIpcCloseMemHandle(p); return rc; }
    w->peer_ipc[shard] = p;
    w->peer_base[shard] = (uint8_t *)p + offset;
    return SHMEMG_OK;
}

extern "C" int shmemg_shard_attach_ptr(shmemg_world_t *w, int shard, void *peer_slab_dev) {
    if (!w || !w->nshards || !peer_slab_dev || shard < 0 || shard >= w->nshards || shard == w->shard) return SHMEMG_ERR_ARG;
    if (w->peer_base[shard]) return SHMEMG_ERR_ARG;
    const int rc = peer_reachable(w, peer_slab_dev);
    if (rc) return rc;
    w->peer_base[shard] = (uint8_t *)peer_slab_dev;
    return SHMEMG_OK;
}

void shmemg_shard_release(shmemg_world *w) {                      // shmemg_finalize
    for (int s = 0; s < SHMEMG_MAX_SHARDS; ++s)
        if (w->peer_ipc[s]) { cudaIpcCloseMemHandle(w->peer_ipc[s]); w->peer_ipc[s] = nullptr; }
}

static int shard_view(const shmemg_world *w, ShardView &v) {
    if (!w || !w->nshards) return SHMEMG_ERR_ARG;
    for (int s = 0; s < w->nshards; ++s) {
        if (!w->peer_base[s]) return SHMEMG_ERR_ARG;             // a shard is not attached yet
        v.base[s] = w->peer_base[s];
    }
    for (int s = w->nshards; s < SHMEMG_MAX_SHARDS; ++s) v.base[s] = nullptr;
    v.stride = w->stride; v.nshards = w->nshards; v.shard = w->shard; v.npes_local = w->npes;
    return SHMEMG_OK;
}
static bool gpe_ok(const shmemg_world *w, int gpe) { return gpe >= 0 && gpe < w->nshards * w->npes; }
static bool gpe_local(const shmemg_world *w, int gpe) { return gpe_ok(w, gpe) && gpe % w->nshards == w->shard; }
static uint8_t *host_g_addr(const shmemg_world *w, int gpe, uint64_t off) {
    return w->peer_base[gpe % w->nshards] + (size_t)(gpe / w->nshards) * w->stride + off;
}

static int launch_shard_copy(shmemg_world *w, uint8_t *dst, const uint8_t *src, size_t nbytes, unsigned long long *sig,
                             uint64_t sig_value, int sig_op, cudaStream_t st) {
    if (nbytes == 0 && !sig) return SHMEMG_OK;
    unsigned *counter = sig ? &w->ctl->sig_counter[(w->sig_seq++) % SHMEMG_SIG_SLOTS] : nullptr;
    const uint64_t maxgrid = (uint64_t)w->sm_count * w->ctas_per_sm;
    uint32_t tb = 8192;
    while (tb < 65536 && nbytes / tb > maxgrid * 8) tb <<= 1;
    const uint64_t ntiles = (nbytes + tb - 1) / tb;
    const uint32_t grid = (uint32_t)(ntiles < maxgrid ? (ntiles ? ntiles : 1) : maxgrid);
    k_shard_copy<<<grid, SHMEMG_THREADS, 0, st>>>(dst, src, nbytes, tb, sig, sig_value, sig_op, counter);
    SHMEMG_CUDA(w, cudaGetLastError());
    return SHMEMG_OK;
}

static int check_transfer(const shmemg_world *w, ShardView &v, uint64_t dest_off, uint64_t source_off, size_t nbytes, int gpe,
                          int target_gpe) {
    int rc = shard_view(w, v);
    if (rc) return rc;
    if (!gpe_local(w, gpe) || !gpe_ok(w, target_gpe)) return SHMEMG_ERR_PE;
    if (!shmemg_in_range(w, dest_off, nbytes) || !shmemg_in_range(w, source_off, nbytes)) return SHMEMG_ERR_RANGE;
    return SHMEMG_OK;
}

// both endpoints on this shard: the single-GPU path (bulk-copy pipeline, GPU-scope signal) does the transfer
static bool both_local(const shmemg_world *w, int target_gpe) { return target_gpe % w->nshards == w->shard; }

extern "C" int shmemg_gput_on_stream(shmemg_world_t *w, uint64_t dest_off, uint64_t source_off, size_t nbytes, int gpe,
                                     int target_gpe, void *stream) {
    ShardView v;
    int rc = check_transfer(w, v, dest_off, source_off, nbytes, gpe, target_gpe);
    if (rc) return rc;
    if (both_local(w, target_gpe))
        return shmemg_put_on_stream(w, dest_off, source_off, nbytes, gpe / w->nshards, target_gpe / w->nshards, stream);
    return launch_shard_copy(w, host_g_addr(w, target_gpe, dest_off), host_g_addr(w, gpe, source_off), nbytes, nullptr, 0, 0,
                             (cudaStream_t)stream);
}
extern "C" int shmemg_gget_on_stream(shmemg_world_t *w, uint64_t dest_off, uint64_t source_off, size_t nbytes, int gpe,
                                     int target_gpe, void *stream) {
    ShardView v;
    int rc = check_transfer(w, v, dest_off, source_off, nbytes, gpe, target_gpe);
    if (rc) return rc;
    if (both_local(w, target_gpe))
        return shmemg_get_on_stream(w, dest_off, source_off, nbytes, gpe / w->nshards, target_gpe / w->nshards, stream);
    return launch_shard_copy(w, host_g_addr(w, gpe, dest_off), host_g_addr(w, target_gpe, source_off), nbytes, nullptr, 0, 0,
                             (cudaStream_t)stream);
}
extern "C" int shmemg_gput_signal_on_stream(shmemg_world_t *w, uint64_t dest_off, uint64_t source_off, size_t nbytes,
                                            uint64_t sig_off, uint64_t signal, int sig_op, int gpe, int target_gpe, void *stream) {
    if (sig_op < SHMEMG_SIGNAL_SET || sig_op > SHMEMG_SIGNAL_ADD) return SHMEMG_ERR_ARG;
    ShardView v;
    int rc = check_transfer(w, v, dest_off, source_off, nbytes, gpe, target_gpe);
    if (rc) return rc;
    if (!shmemg_in_range(w, sig_off, 8)) return SHMEMG_ERR_RANGE;
    if (sig_off & 7) return SHMEMG_ERR_ALIGN;
    // a signal word may also be updated from another shard (system scope): only a one-shard world takes the GPU-scope path
    if (w->nshards == 1)
        return shmemg_put_signal_on_stream(w, dest_off, source_off, nbytes, sig_off, signal, sig_op, gpe / w->nshards,
                                           target_gpe / w->nshards, stream);
    return launch_shard_copy(w, host_g_addr(w, target_gpe, dest_off), host_g_addr(w, gpe, source_off), nbytes,
                             (unsigned long long *)host_g_addr(w, target_gpe, sig_off), signal, sig_op, (cudaStream_t)stream);
}
extern "C" int shmemg_gsignal_wait_until_on_stream(shmemg_world_t *w, uint64_t sig_off, int cmp, uint64_t value, int gpe,
                                                   void *stream) {
    ShardView v;
    int rc = shard_view(w, v);
    if (rc) return rc;
    if (cmp < SHMEMG_CMP_EQ || cmp > SHMEMG_CMP_LE) return SHMEMG_ERR_ARG;
    if (!gpe_local(w, gpe)) return SHMEMG_ERR_PE;
    if (!shmemg_in_range(w, sig_off, 8)) return SHMEMG_ERR_RANGE;
    if (sig_off & 7) return SHMEMG_ERR_ALIGN;
    k_shard_wait_until<<<1, 1, 0, (cudaStream_t)stream>>>((const unsigned long long *)host_g_addr(w, gpe, sig_off), cmp, value);
    SHMEMG_CUDA(w, cudaGetLastError());
    return SHMEMG_OK;
}

template <int OP>
static int launch_shard_amo(shmemg_world *w, const ShardAmoArgs &a, int idx_bytes, cudaStream_t st) {
    size_t blocks = (a.n + 255) / 256;
    const size_t cap = (size_t)w->sm_count * 8 * 4;
    if (blocks > cap) blocks = cap;
    if (idx_bytes == 4) k_shard_amo<4, OP><<<(unsigned)blocks, 256, 0, st>>>(a);
    else k_shard_amo<8, OP><<<(unsigned)blocks, 256, 0, st>>>(a);
    SHMEMG_CUDA(w, cudaGetLastError());
    return SHMEMG_OK;
}

extern "C" int shmemg_gatomic_batch_on_stream(shmemg_world_t *w, int op, uint64_t sym_off, const int32_t *target_gpe,
                                              const void *elem_idx, int idx_bytes, const uint64_t *cond, uint64_t cond_scalar,
                                              const uint64_t *val, uint64_t val_scalar, uint64_t *fetched_out, size_t n,
                                              void *stream) {
    ShardAmoArgs a;
    int rc = shard_view(w, a.v);
    if (rc) return rc;
    if (op < SHMEMG_OP_ATOMIC_ADD || op > SHMEMG_OP_ATOMIC_COMPARE_SWAP) return SHMEMG_ERR_ARG;
    if (n && (!target_gpe || !elem_idx)) return SHMEMG_ERR_ARG;
    if (idx_bytes != 4 && idx_bytes != 8) return SHMEMG_ERR_ARG;
    if (op != SHMEMG_OP_ATOMIC_ADD && n && !fetched_out) return SHMEMG_ERR_ARG;
    if (sym_off & 7) return SHMEMG_ERR_ALIGN;
    if (!shmemg_in_range(w, sym_off, 8)) return SHMEMG_ERR_RANGE;
    if (n == 0) return SHMEMG_OK;
    // target_gpe[] and elem_idx[] are DEVICE arrays: per-op bounds are the caller's contract (undefined otherwise)
    a.sym_off = sym_off; a.tgt = target_gpe; a.idx = elem_idx;
    a.val = (const unsigned long long *)val; a.cond = (const unsigned long long *)cond;
    a.val_s = val_scalar; a.cond_s = cond_scalar; a.fetched = (unsigned long long *)fetched_out; a.n = n;
    cudaStream_t st = (cudaStream_t)stream;
    if (op == SHMEMG_OP_ATOMIC_ADD) return launch_shard_amo<SHMEMG_OP_ATOMIC_ADD>(w, a, idx_bytes, st);
    if (op == SHMEMG_OP_ATOMIC_FETCH_ADD) return launch_shard_amo<SHMEMG_OP_ATOMIC_FETCH_ADD>(w, a, idx_bytes, st);
    return launch_shard_amo<SHMEMG_OP_ATOMIC_COMPARE_SWAP>(w, a, idx_bytes, st);
}

extern "C" int shmemg_galltoall_on_stream(shmemg_world_t *w, uint64_t dest_off, uint64_t source_off, size_t nbytes_per_pe,
                                          void *stream) {
    ShardView v;
    int rc = shard_view(w, v);
    if (rc) return rc;
    const uint64_t gn = (uint64_t)w->nshards * w->npes;
    if (nbytes_per_pe && gn > w->heap_bytes / nbytes_per_pe) return SHMEMG_ERR_RANGE;
    const uint64_t span = gn * nbytes_per_pe;
    if (!shmemg_in_range(w, dest_off, span) || !shmemg_in_range(w, source_off, span)) return SHMEMG_ERR_RANGE;
    if (nbytes_per_pe == 0) return SHMEMG_OK;
    if (dest_off < source_off + span && source_off < dest_off + span) return SHMEMG_ERR_OVERLAP;
    if (((dest_off | source_off | nbytes_per_pe | w->stride) & 15) == 0) {
        if (!w->smem_attr_shard) {
            SHMEMG_CUDA(w, cudaFuncSetAttribute(k_shard_alltoall_tma, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SHMEMG_TMA_SMEM));
            w->smem_attr_shard = true;
        }
        const uint64_t it = (uint64_t)w->npes * gn * ((nbytes_per_pe + SHMEMG_TMA_TILE - 1) / SHMEMG_TMA_TILE);
        k_shard_alltoall_tma<<<(unsigned)(it < (uint64_t)w->sm_count ? it : (uint64_t)w->sm_count), 32, SHMEMG_TMA_SMEM,
                               (cudaStream_t)stream>>>(v, dest_off, source_off, nbytes_per_pe);
        SHMEMG_CUDA(w, cudaGetLastError());
        return SHMEMG_OK;
    }
    const unsigned chunk = 32768;
    const uint64_t items = (uint64_t)w->npes * gn * ((nbytes_per_pe + chunk - 1) / chunk);
    const uint64_t maxgrid = (uint64_t)w->sm_count * w->ctas_per_sm;
    k_shard_alltoall<<<(unsigned)(items < maxgrid ? items : maxgrid), SHMEMG_THREADS, 0, (cudaStream_t)stream>>>(
        v, dest_off, source_off, nbytes_per_pe, chunk);
    SHMEMG_CUDA(w, cudaGetLastError());
    return SHMEMG_OK;
}

extern "C" int shmemg_gfcollect_on_stream(shmemg_world_t *w, uint64_t dest_off, uint64_t source_off, size_t nbytes, void *stream) {
    ShardView v;
    int rc = shard_view(w, v);
    if (rc) return rc;
    const uint64_t gn = (uint64_t)w->nshards * w->npes;
    if (nbytes && gn > w->heap_bytes / nbytes) return SHMEMG_ERR_RANGE;
    const uint64_t span = gn * nbytes;
    if (!shmemg_in_range(w, dest_off, span) || !shmemg_in_range(w, source_off, nbytes)) return SHMEMG_ERR_RANGE;
    if (nbytes == 0) return SHMEMG_OK;
    if (dest_off < source_off + nbytes && source_off < dest_off + span) return SHMEMG_ERR_OVERLAP;
    const unsigned chunk = 32768;
    const uint64_t items = (uint64_t)w->npes * gn * ((nbytes + chunk - 1) / chunk);
    const uint64_t maxgrid = (uint64_t)w->sm_count * w->ctas_per_sm;
    k_shard_fcollect<<<(unsigned)(items < maxgrid ? items : maxgrid), SHMEMG_THREADS, 0, (cudaStream_t)stream>>>(v, dest_off, source_off,
                                                                                                               nbytes, chunk);
    SHMEMG_CUDA(w, cudaGetLastError());
    return SHMEMG_OK;
}

extern "C" int shmemg_gsum_reduce_on_stream(shmemg_world_t *w, int dtype, uint64_t dest_off, uint64_t source_off, size_t nreduce,
                                            void *stream) {
    ShardView v;
    int rc = shard_view(w, v);
    if (rc) return rc;
    if (dtype != SHMEMG_F32 && dtype != SHMEMG_I64) return SHMEMG_ERR_ARG;
    const size_t es = dtype == SHMEMG_F32 ? 4 : 8;
    if (nreduce > w->heap_bytes / es) return SHMEMG_ERR_RANGE;
    const uint64_t span = (uint64_t)nreduce * es;
    if (!shmemg_in_range(w, dest_off, span) || !shmemg_in_range(w, source_off, span)) return SHMEMG_ERR_RANGE;
    if ((dest_off | source_off) & (es - 1)) return SHMEMG_ERR_ALIGN;
    if (nreduce == 0) return SHMEMG_OK;
    if (dest_off < source_off + span && source_off < dest_off + span) return SHMEMG_ERR_OVERLAP;
    // this shard's share: elements [e0, e1), cut at multiples of 32 elements
    const size_t per = ((nreduce + (size_t)w->nshards - 1) / (size_t)w->nshards + 31) / 32 * 32;
    const size_t e0 = per * (size_t)w->shard < nreduce ? per * (size_t)w->shard : nreduce;
    const size_t e1 = e0 + per < nreduce ? e0 + per : nreduce;
    if (e1 == e0) return SHMEMG_OK;
    const uint64_t maxgrid = (uint64_t)w->sm_count * 8;
    const uint64_t blocks = (e1 - e0 + 255) / 256;
    const unsigned grid = (unsigned)(blocks < maxgrid ? blocks : maxgrid);
    if (dtype == SHMEMG_F32) k_shard_sum_reduce<float><<<grid, 256, 0, (cudaStream_t)stream>>>(v, dest_off, source_off, e0, e1);
    else k_shard_sum_reduce<long long><<<grid, 256, 0, (cudaStream_t)stream>>>(v, dest_off, source_off, e0, e1);
    SHMEMG_CUDA(w, cudaGetLastError());
    return SHMEMG_OK;
}

extern "C" int shmemg_gbarrier_all_on_stream(shmemg_world_t *w, void *stream) {
    ShardView v;
    int rc = shard_view(w, v);
    if (rc) return rc;
    const unsigned long long ctl_off = (unsigned long long)((uint8_t *)w->ctl - w->base);
    const unsigned long long bar_off = (unsigned long long)offsetof(CtlRegion, shard_bar);
    k_shard_barrier<<<1, 32, 0, (cudaStream_t)stream>>>(v, ctl_off, bar_off, ++w->shard_epoch);
    SHMEMG_CUDA(w, cudaGetLastError());
    return SHMEMG_OK;
}
