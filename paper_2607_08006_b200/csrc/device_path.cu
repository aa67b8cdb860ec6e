// device_path.cu -- the DEVICE-INITIATED path (Tier-1): kernels that issue the specification's
// operations themselves through the header-only entry points of include/shmemg_device.cuh.
//   k_device_exec_ops : one thread block per PE ("PE agent", cooperative launch); agent p walks an op list in order and
//                       executes the ops it initiates with blocking semantics.  It is the device-side counterpart of
//                       the batch executor and lets every litmus program and parity comparison of the tests run device-initiated.
//   k_halo_persistent : the halo application as ONE persistent kernel (perturb, pack, put_signal, wait for all rounds),
//                       see halo_app.cu for the host-driven version of the same application.
#include "internal.cuh"
#include "../../include/shmemg_device.cuh"
#include "../../include/shmemg_app.h"

extern "C" int shmemg_device_world_get(const shmemg_world_t *w, shmemg_device_world_t *out) {
    if (!w || !out) return SHMEMG_ERR_ARG;
    out->base = w->base;
    out->stride = w->stride;
    out->heap_bytes = w->heap_bytes;
    out->npes = w->npes;
    out->reserved = 0;
    out->bar_arrivals = &w->ctl->bar_arrivals;
    out->reserved2 = nullptr;
    return SHMEMG_OK;
}

#define AGENT_THREADS 256

__device__ __forceinline__ shmemg_op_t ld_op(const shmemg_op_t *p) {
    shmemg_op_t r;
    const int4 *s = reinterpret_cast<const int4 *>(p);
    int4 *d = reinterpret_cast<int4 *>(&r);
    d[0] = __ldg(s); d[1] = __ldg(s + 1); d[2] = __ldg(s + 2); d[3] = __ldg(s + 3);
    return r;
}

__global__ void __launch_bounds__(AGENT_THREADS) k_device_exec_ops(const shmemg_device_world_t dw, const shmemg_op_t *ops,
                                                                   size_t nops) {
    const int p = blockIdx.x;                       // this block acts for PE p
    for (size_t i = 0; i < nops; ++i) {
        const shmemg_op_t o = ld_op(ops + i);       // every thread reads the same descriptor: uniform participation
        if (o.opcode == SHMEMG_OP_BARRIER_ALL) { shmemg_dev_barrier_all_block(dw); continue; }
        if (o.initiator_pe != p) continue;
        switch (o.opcode) {
        case SHMEMG_OP_PUT:
            shmemg_dev_put_block(dw, o.rem_off, o.loc_off, o.nbytes, p, o.target_pe);
            break;
        case SHMEMG_OP_GET:
            shmemg_dev_get_block(dw, o.loc_off, o.rem_off, o.nbytes, p, o.target_pe);
            break;
        case SHMEMG_OP_PUT_SIGNAL:
            shmemg_dev_put_signal_block(dw, o.rem_off, o.loc_off, o.nbytes, o.sig_off, o.value, o.sig_op, p, o.target_pe);
            break;
        case SHMEMG_OP_ATOMIC_ADD:
            if (threadIdx.x == 0) shmemg_dev_atomic_add(dw, o.rem_off, o.value, o.target_pe);
            break;
        case SHMEMG_OP_ATOMIC_FETCH_ADD:
            if (threadIdx.x == 0)
                *reinterpret_cast<unsigned long long *>(shmemg_dev_ptr(dw, o.loc_off, p)) =
                    shmemg_dev_atomic_fetch_add(dw, o.rem_off, o.value, o.target_pe);
            __syncthreads();                        // the fetch slot is local state of the agent: later ops may read it
            break;
        case SHMEMG_OP_ATOMIC_COMPARE_SWAP:
            if (threadIdx.x == 0)
                *reinterpret_cast<unsigned long long *>(shmemg_dev_ptr(dw, o.loc_off, p)) =
                    shmemg_dev_atomic_compare_swap(dw, o.rem_off, o.cond, o.value, o.target_pe);
            __syncthreads();
            break;
        case SHMEMG_OP_SIGNAL_WAIT_UNTIL:
            shmemg_dev_signal_wait_until_block(dw, o.loc_off, o.cmp, o.value, p);
            break;
        case SHMEMG_OP_FENCE:
            shmemg_dev_fence_block();
            break;
        case SHMEMG_OP_QUIET:
            shmemg_dev_quiet_block();
            break;
        default: break;
        }
    }
}

extern "C" int shmemg_device_exec_ops_on_stream(shmemg_world_t *w, const shmemg_op_t *ops_host, size_t nops, void *ops_dev,
                                                void *stream, size_t *bad_index) {
    if (!w || (!ops_host && nops) || (!ops_dev && nops)) return SHMEMG_ERR_ARG;
    for (size_t i = 0; i < nops; ++i) {
        int rc = shmemg_validate_op(w, ops_host[i]);
        if (rc) {
            if (bad_index) *bad_index = i;
            return rc;
        }
    }
    if (nops == 0) return SHMEMG_OK;
    int per_sm = 0;
    SHMEMG_CUDA(w, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_device_exec_ops, AGENT_THREADS, 0));
    if ((long long)per_sm * w->sm_count < w->npes) return SHMEMG_ERR_NOMEM;     // agents could not all be co-resident
    cudaStream_t st = (cudaStream_t)stream;
    SHMEMG_CUDA(w, cudaMemcpyAsync(ops_dev, ops_host, nops * sizeof(shmemg_op_t), cudaMemcpyHostToDevice, st));
    shmemg_device_world_t dw;
    shmemg_device_world_get(w, &dw);
    const shmemg_op_t *od = reinterpret_cast<const shmemg_op_t *>(ops_dev);
    void *args[] = {&dw, &od, &nops};
    SHMEMG_CUDA(w, cudaLaunchCooperativeKernel((void *)k_device_exec_ops, dim3((unsigned)w->npes), dim3(AGENT_THREADS), args, 0, st));
    return SHMEMG_OK;
}


// ---- one device collective, device-initiated: one thread block per PE calls the block-scope routine of shmemg_device.cuh ----
#define COLL_THREADS 1024
__global__ void __launch_bounds__(COLL_THREADS) k_device_collective(const shmemg_device_world_t dw, int kind, int dtype, uint64_t dest_off,
                                                                    uint64_t source_off, size_t n, int root) {
    const int p = blockIdx.x;
    switch (kind) {
    case SHMEMG_DEVCOLL_SUM_REDUCE: shmemg_dev_sum_reduce_block(dw, dtype, dest_off, source_off, n, p); break;
    case SHMEMG_DEVCOLL_FCOLLECT: shmemg_dev_fcollect_block(dw, dest_off, source_off, n, p); break;
    case SHMEMG_DEVCOLL_ALLTOALL: shmemg_dev_alltoall_block(dw, dest_off, source_off, n, p); break;
    default: shmemg_dev_broadcast_block(dw, dest_off, source_off, n, root, p); break;
    }
}

extern "C" int shmemg_device_collective_on_stream(shmemg_world_t *w, int kind, int dtype, uint64_t dest_off, uint64_t source_off,
                                                  size_t n, int root, void *stream) {
    if (!w || kind < SHMEMG_DEVCOLL_SUM_REDUCE || kind > SHMEMG_DEVCOLL_BROADCAST) return SHMEMG_ERR_ARG;
    uint64_t dbytes = n, sbytes = n;
    if (kind == SHMEMG_DEVCOLL_SUM_REDUCE) {
        if (dtype < SHMEMG_F32 || dtype > SHMEMG_F64) return SHMEMG_ERR_ARG;
        const uint64_t esz = (dtype == SHMEMG_F32 || dtype == SHMEMG_I32) ? 4 : 8;
        dbytes = sbytes = (uint64_t)n * esz;
        if ((dest_off | source_off) & (esz - 1)) return SHMEMG_ERR_ALIGN;
    } else if (kind == SHMEMG_DEVCOLL_FCOLLECT) {
        dbytes = (uint64_t)n * w->npes;
    } else if (kind == SHMEMG_DEVCOLL_ALLTOALL) {
        dbytes = sbytes = (uint64_t)n * w->npes;
    } else if (!shmemg_pe_ok(w, root)) {
        return SHMEMG_ERR_PE;
    }
    if (!shmemg_in_range(w, dest_off, dbytes) || !shmemg_in_range(w, source_off, sbytes)) return SHMEMG_ERR_RANGE;
    if (n == 0) return SHMEMG_OK;
    const bool overlap = dest_off < source_off + sbytes && source_off < dest_off + dbytes;
    if (overlap && !(kind == SHMEMG_DEVCOLL_SUM_REDUCE && dest_off == source_off)) return SHMEMG_ERR_OVERLAP;
    int per_sm = 0;
    SHMEMG_CUDA(w, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_device_collective, COLL_THREADS, 0));
    if ((long long)per_sm * w->sm_count < w->npes) return SHMEMG_ERR_NOMEM;
    shmemg_device_world_t dw;
    shmemg_device_world_get(w, &dw);
    void *args[] = {&dw, &kind, &dtype, &dest_off, &source_off, &n, &root};
    SHMEMG_CUDA(w, cudaLaunchCooperativeKernel((void *)k_device_collective, dim3((unsigned)w->npes), dim3(COLL_THREADS), args, 0,
                                               (cudaStream_t)stream));
    return SHMEMG_OK;
}


// ---- explicit device contexts (NEXT-3) ------------------------------------------------------------------------------------
extern "C" size_t shmemg_ctx_bytes(uint32_t queue_entries) {
    if (queue_entries == 0) return 0;
    return 256 + (size_t)queue_entries * sizeof(shmemg_nbi_rec_t);
}
extern "C" int shmemg_ctx_create(shmemg_world_t *w, int pe, uint32_t queue_entries, void *ctx_mem_dev, size_t ctx_mem_bytes,
                                 void *stream, shmemg_device_ctx_t *out) {
    if (!w || !out || !ctx_mem_dev || queue_entries == 0) return SHMEMG_ERR_ARG;
    if (!shmemg_pe_ok(w, pe)) return SHMEMG_ERR_PE;
    if ((uintptr_t)ctx_mem_dev % 256) return SHMEMG_ERR_ALIGN;
    if (ctx_mem_bytes < shmemg_ctx_bytes(queue_entries)) return SHMEMG_ERR_NOMEM;
    SHMEMG_CUDA(w, cudaMemsetAsync(ctx_mem_dev, 0, 256, (cudaStream_t)stream));
    out->counters = (unsigned long long *)ctx_mem_dev;
    out->queue = (shmemg_nbi_rec_t *)((uint8_t *)ctx_mem_dev + 256);
    out->capacity = queue_entries;
    out->pe = pe;
    return SHMEMG_OK;
}
extern "C" int shmemg_ctx_counters(shmemg_world_t *w, const shmemg_device_ctx_t *ctx, void *stream, uint64_t *issued, uint64_t *completed) {
    if (!w || !ctx || !ctx->counters) return SHMEMG_ERR_ARG;
    unsigned long long v[2] = {0, 0};
    SHMEMG_CUDA(w, cudaMemcpyAsync(v, ctx->counters, 16, cudaMemcpyDeviceToHost, (cudaStream_t)stream));
    SHMEMG_CUDA(w, cudaStreamSynchronize((cudaStream_t)stream));
    if (issued) *issued = v[0];
    if (completed) *completed = v[1];
    return SHMEMG_OK;
}

// the PE-agent interpreter with explicit contexts: PUT / GET / PUT_SIGNAL are non-blocking on the op's context
__global__ void __launch_bounds__(AGENT_THREADS) k_device_exec_ops_ctx(const shmemg_device_world_t dw, const shmemg_op_t *ops, size_t nops,
                                                                       const shmemg_device_ctx_t *ctxs, int nctx, unsigned flags) {
    const int p = blockIdx.x;
    const shmemg_device_ctx_t *mine = ctxs + (size_t)p * nctx;
    auto progress_all = [&]() { for (int c = 0; c < nctx; ++c) shmemg_dev_ctx_quiet_block(mine[c]); };
    for (size_t i = 0; i < nops; ++i) {
        const shmemg_op_t o = ld_op(ops + i);
        if (o.opcode == SHMEMG_OP_BARRIER_ALL) { progress_all(); shmemg_dev_barrier_all_block(dw); continue; }   // barrier implies quiet
        if (o.initiator_pe != p) continue;
        const shmemg_device_ctx_t c = mine[o.ctx];
        switch (o.opcode) {
        case SHMEMG_OP_PUT:
            if (threadIdx.x == 0) shmemg_dev_put_nbi(dw, c, o.rem_off, o.loc_off, o.nbytes, o.target_pe);
            __syncthreads();
            break;
        case SHMEMG_OP_GET:
            if (threadIdx.x == 0) shmemg_dev_get_nbi(dw, c, o.loc_off, o.rem_off, o.nbytes, o.target_pe);
            __syncthreads();
            break;
        case SHMEMG_OP_PUT_SIGNAL:
            if (threadIdx.x == 0) shmemg_dev_put_signal_nbi(dw, c, o.rem_off, o.loc_off, o.nbytes, o.sig_off, o.value, o.sig_op, o.target_pe);
            __syncthreads();
            break;
        case SHMEMG_OP_ATOMIC_ADD:
            if (threadIdx.x == 0) shmemg_dev_atomic_add(dw, o.rem_off, o.value, o.target_pe);
            break;
        case SHMEMG_OP_ATOMIC_FETCH_ADD:
            if (threadIdx.x == 0)
                *reinterpret_cast<unsigned long long *>(shmemg_dev_ptr(dw, o.loc_off, p)) =
                    shmemg_dev_atomic_fetch_add(dw, o.rem_off, o.value, o.target_pe);
            __syncthreads();
            break;
        case SHMEMG_OP_ATOMIC_COMPARE_SWAP:
            if (threadIdx.x == 0)
                *reinterpret_cast<unsigned long long *>(shmemg_dev_ptr(dw, o.loc_off, p)) =
                    shmemg_dev_atomic_compare_swap(dw, o.rem_off, o.cond, o.value, o.target_pe);
            __syncthreads();
            break;
        case SHMEMG_OP_SIGNAL_WAIT_UNTIL:
            progress_all();                         // a PE that blocks first progresses its pending operations (no deadlock)
            shmemg_dev_signal_wait_until_block(dw, o.loc_off, o.cmp, o.value, p);
            break;
        case SHMEMG_OP_FENCE:
            shmemg_dev_fence_gpu();                 // the AMOs issued at once
            shmemg_dev_ctx_fence_block(c);
            break;
        case SHMEMG_OP_QUIET:
            shmemg_dev_fence_gpu();
            shmemg_dev_ctx_quiet_block(c);
            break;
        default: break;
        }
    }
    if (!(flags & SHMEMG_EXEC_LEAVE_PENDING)) progress_all();     // end of the list = quiet for every context
}

extern "C" int shmemg_device_exec_ops_ctx_on_stream(shmemg_world_t *w, const shmemg_op_t *ops_host, size_t nops, void *ops_dev,
                                                    const shmemg_device_ctx_t *ctxs_dev, int nctx, uint32_t flags, void *stream,
                                                    size_t *bad_index) {
    if (!w || (!ops_host && nops) || (!ops_dev && nops) || !ctxs_dev || nctx < 1 || nctx > SHMEMG_CTX_MAX) return SHMEMG_ERR_ARG;
    for (size_t i = 0; i < nops; ++i) {
        int rc = shmemg_validate_op(w, ops_host[i]);
        if (!rc && ops_host[i].opcode != SHMEMG_OP_BARRIER_ALL && ops_host[i].ctx >= nctx) rc = SHMEMG_ERR_ARG;
        if (rc) {
            if (bad_index) *bad_index = i;
            return rc;
        }
    }
    if (nops == 0) return SHMEMG_OK;
    int per_sm = 0;
    SHMEMG_CUDA(w, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_device_exec_ops_ctx, AGENT_THREADS, 0));
    if ((long long)per_sm * w->sm_count < w->npes) return SHMEMG_ERR_NOMEM;
    cudaStream_t st = (cudaStream_t)stream;
    SHMEMG_CUDA(w, cudaMemcpyAsync(ops_dev, ops_host, nops * sizeof(shmemg_op_t), cudaMemcpyHostToDevice, st));
    shmemg_device_world_t dw;
    shmemg_device_world_get(w, &dw);
    const shmemg_op_t *od = reinterpret_cast<const shmemg_op_t *>(ops_dev);
    void *args[] = {&dw, &od, &nops, &ctxs_dev, &nctx, &flags};
    SHMEMG_CUDA(w, cudaLaunchCooperativeKernel((void *)k_device_exec_ops_ctx, dim3((unsigned)w->npes), dim3(AGENT_THREADS), args, 0, st));
    return SHMEMG_OK;
}
