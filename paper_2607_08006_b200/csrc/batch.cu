// batch.cu -- op-batch planner (host) and the persistent-grid batch executor kernel (sm_100a),
// plus the single put/get/put_signal/wait `_on_stream` calls.  SURVEY.md 8(a) rows a5-a8, a12-a14.
//
// Executor design:
//   * the host planner resolves PE->address translation, cuts copy ops into tiles and groups consecutive
//     AMO descriptors into runs; tiles are listed in batch order;
//   * a persistent grid claims tiles with one global ticket IN BATCH ORDER, so a claimed tile only ever
//     waits for tiles with smaller tickets, which are finished or held by running CTAs: no deadlock and no
//     co-residency requirement;
//   * ordering state: done[p] = completed ops of PE p, done[npes] = completed ops of all PEs (monotonic,
//     release-incremented).  An op that follows a FENCE/QUIET/WAIT of its PE starts only when done[p] has
//     reached the number of that PE's ops before the marker; an op after a BARRIER_ALL starts only when
//     done[npes] has reached the number of ops before the barrier (acquire spin by one thread + bar.sync);
//   * a multi-tile op completes at its last-arriving tile (fence + relaxed counter), which then performs
//     the put_signal update with release semantics and the done[] increments.
#include <stdlib.h>
#include <string.h>

#include <vector>

#include "internal.cuh"

#define AMO_RUN_MAX SHMEMG_THREADS
#define OPF_COUNT_PE 0x10000u    // a later marker of this PE depends on this op: bump done[initiator]
#define OPF_COUNT_ALL 0x20000u   // a later BARRIER_ALL depends on this op: bump done[npes]

struct DevOp {            // 64 B, resolved on the host
    uint64_t dst;         // copy destination / AMO target word
    uint64_t src;         // copy source / AMO fetch slot (0 = none)
    uint64_t nbytes;
    uint64_t sig;         // put_signal: signal word on the target; wait: the local word
    uint64_t value;
    uint64_t cond;
    uint32_t kind;        // bits 0-7 opcode, 8-15 sig_op or cmp, 16+ OPF_*
    uint32_t initiator;
    uint32_t dep_pe;      // start when done[initiator] >= dep_pe
    uint32_t dep_all;     // and done[npes] >= dep_all
};
static_assert(sizeof(DevOp) == 64, "DevOp must be 64 bytes");

struct Tile { uint32_t op; uint32_t sub; };   // copy/wait: sub = tile index within op; AMO run: sub = count

struct PlanHeader {       // 256 B at the start of the plan buffer
    uint32_t ntiles, nops, npes, tile_bytes;
    uint32_t ticket, exited, pad0, pad1;
    uint64_t ops_off, tiles_off, done_off, arrive_off;
    uint64_t pad2[24];
};
static_assert(sizeof(PlanHeader) == 256, "PlanHeader must be 256 bytes");

struct shmemg_batch {
    shmemg_world *w;
    uint8_t *plan_dev;
    uint32_t ntiles;
    uint32_t grid;
};

// ---------------------------------------------------------------------------------------------------------
// device
// ---------------------------------------------------------------------------------------------------------
__device__ __forceinline__ void wait_deps(const unsigned *done, unsigned npes, unsigned initiator, unsigned dep_pe,
                                          unsigned dep_all) {
    if (dep_pe) while (ld_acquire_u32(done + initiator) < dep_pe) __nanosleep(32);
    if (dep_all) while (ld_acquire_u32(done + npes) < dep_all) __nanosleep(32);
}

__device__ __forceinline__ void count_done(unsigned *done, unsigned npes, unsigned kind, unsigned initiator) {
    if (kind & OPF_COUNT_PE) red_release_add_u32(done + initiator, 1u);
    if (kind & OPF_COUNT_ALL) red_release_add_u32(done + npes, 1u);
}

__device__ __forceinline__ void amo_one(const DevOp &o) {
    unsigned long long *word = reinterpret_cast<unsigned long long *>(o.dst);
    const unsigned opc = o.kind & 0xffu;
    if (opc == SHMEMG_OP_ATOMIC_ADD) {
        asm volatile("red.relaxed.gpu.global.add.u64 [%0], %1;" ::"l"(word), "l"(o.value) : "memory");
    } else if (opc == SHMEMG_OP_ATOMIC_FETCH_ADD) {
        unsigned long long old = atomicAdd(word, (unsigned long long)o.value);
        *reinterpret_cast<volatile unsigned long long *>(o.src) = old;
    } else {
        unsigned long long old = atomicCAS(word, (unsigned long long)o.cond, (unsigned long long)o.value);
        *reinterpret_cast<volatile unsigned long long *>(o.src) = old;
    }
}

__global__ void __launch_bounds__(SHMEMG_THREADS, 4) k_batch_exec(uint8_t *plan) {
    PlanHeader *hdr = reinterpret_cast<PlanHeader *>(plan);
    const DevOp *__restrict__ ops = reinterpret_cast<const DevOp *>(plan + hdr->ops_off);
    const Tile *__restrict__ tiles = reinterpret_cast<const Tile *>(plan + hdr->tiles_off);
    unsigned *done = reinterpret_cast<unsigned *>(plan + hdr->done_off);
    unsigned *arrive = reinterpret_cast<unsigned *>(plan + hdr->arrive_off);
    const unsigned ntiles = hdr->ntiles, npes = hdr->npes, tile_bytes = hdr->tile_bytes;
    const int tid = threadIdx.x;
    __shared__ unsigned s_ticket;
    __shared__ unsigned s_last;

    if (tid == 0) s_ticket = atomicAdd(&hdr->ticket, 1u);
    __syncthreads();
    unsigned t = s_ticket;
    while (t < ntiles) {
        unsigned next = 0;
        if (tid == 0) next = atomicAdd(&hdr->ticket, 1u);     // claim ahead: hides the L2 round trip
        const Tile tl = tiles[t];
        const unsigned kind0 = ops[tl.op].kind;
        const unsigned opc = kind0 & 0xffu;
        if (opc <= SHMEMG_OP_PUT_SIGNAL) {
            // ---- copy tile -------------------------------------------------------------------------------
            const DevOp o = ops[tl.op];
            if (o.dep_pe | o.dep_all) {
                if (tid == 0) wait_deps(done, npes, o.initiator, o.dep_pe, o.dep_all);
                __syncthreads();
            }
            const uint64_t off = (uint64_t)tl.sub * tile_bytes;
            uint64_t n = o.nbytes - off;
            if (n > tile_bytes) n = tile_bytes;
            copy_coop<8>(reinterpret_cast<uint8_t *>(o.dst + off), reinterpret_cast<const uint8_t *>(o.src + off), n,
                         tid, SHMEMG_THREADS);
            __syncthreads();                                   // every thread's stores precede thread 0's release
            if (tid == 0) {
                const unsigned nt = o.nbytes <= tile_bytes ? 1u : (unsigned)((o.nbytes + tile_bytes - 1) / tile_bytes);
                bool last = true;
                if (nt > 1) {
                    __threadfence();
                    last = (atomicAdd(arrive + tl.op, 1u) == nt - 1);
                    if (last) __threadfence();
                }
                if (last) {
                    if (opc == SHMEMG_OP_PUT_SIGNAL)
                        signal_update(reinterpret_cast<unsigned long long *>(o.sig), o.value, (o.kind >> 8) & 0xff);
                    count_done(done, npes, o.kind, o.initiator);
                }
                s_ticket = next;
            }
        } else if (opc == SHMEMG_OP_SIGNAL_WAIT_UNTIL) {
            if (tid == 0) {
                const DevOp o = ops[tl.op];
                wait_deps(done, npes, o.initiator, o.dep_pe, o.dep_all);
                const unsigned long long *sig = reinterpret_cast<const unsigned long long *>(o.sig);
                const int cmp = (o.kind >> 8) & 0xff;
                while (!cmp_u64(cmp, ld_acquire_u64(sig), o.value)) __nanosleep(64);
                count_done(done, npes, o.kind, o.initiator);
                s_ticket = next;
            }
        } else {
            // ---- run of AMO descriptors: one thread per op ---------------------------------------------
            if (tid < (int)tl.sub) {
                const DevOp o = ops[tl.op + tid];
                wait_deps(done, npes, o.initiator, o.dep_pe, o.dep_all);
                amo_one(o);
                count_done(done, npes, o.kind, o.initiator);
            }
            if (tid == 0) s_ticket = next;
        }
        __syncthreads();
        t = s_ticket;
        __syncthreads();                                       // nobody overwrites s_ticket before all have read it
    }
    // last CTA out re-arms the plan so the batch can be enqueued again
    if (tid == 0) s_last = (atomicAdd(&hdr->exited, 1u) == gridDim.x - 1);
    __syncthreads();
    if (s_last) {
        for (unsigned i = tid; i <= npes; i += SHMEMG_THREADS) done[i] = 0;
        for (unsigned i = tid; i < hdr->nops; i += SHMEMG_THREADS) arrive[i] = 0;
        if (tid == 0) { hdr->ticket = 0; hdr->exited = 0; }
    }
}

// single copy on a stream: grid-stride over tiles, optional last-arriver signal
__global__ void __launch_bounds__(SHMEMG_THREADS, 4)
k_copy_single(uint8_t *dst, const uint8_t *src, size_t nbytes, unsigned tile_bytes, unsigned long long *sig,
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
            __threadfence();
            if (atomicAdd(counter, 1u) == gridDim.x - 1) {
                __threadfence();
                *counter = 0;
                signal_update(sig, sig_value, sig_op);
            }
        }
    }
}

__global__ void k_wait_until(const unsigned long long *sig, int cmp, unsigned long long value) {
    while (!cmp_u64(cmp, ld_acquire_u64(sig), value)) __nanosleep(100);
}

// ---------------------------------------------------------------------------------------------------------
// host: validation + planning
// ---------------------------------------------------------------------------------------------------------
static int validate_op(const shmemg_world *w, const shmemg_op_t &o) {
    switch (o.opcode) {
    case SHMEMG_OP_FENCE: case SHMEMG_OP_QUIET:
        return shmemg_pe_ok(w, o.initiator_pe) ? SHMEMG_OK : SHMEMG_ERR_PE;
    case SHMEMG_OP_BARRIER_ALL:
        return SHMEMG_OK;
    default: break;
    }
    if (o.opcode < SHMEMG_OP_PUT || o.opcode > SHMEMG_OP_BARRIER_ALL) return SHMEMG_ERR_ARG;
    if (!shmemg_pe_ok(w, o.initiator_pe)) return SHMEMG_ERR_PE;
    if (o.opcode == SHMEMG_OP_SIGNAL_WAIT_UNTIL) {
        if (o.cmp > SHMEMG_CMP_LE) return SHMEMG_ERR_ARG;
        if (!shmemg_in_range(w, o.loc_off, 8)) return SHMEMG_ERR_RANGE;
        return (o.loc_off & 7) ? SHMEMG_ERR_ALIGN : SHMEMG_OK;
    }
    if (!shmemg_pe_ok(w, o.target_pe)) return SHMEMG_ERR_PE;
    if (o.opcode <= SHMEMG_OP_PUT_SIGNAL) {
        if (!shmemg_in_range(w, o.rem_off, o.nbytes) || !shmemg_in_range(w, o.loc_off, o.nbytes)) return SHMEMG_ERR_RANGE;
        if (o.opcode == SHMEMG_OP_PUT_SIGNAL) {
            if (o.sig_op > SHMEMG_SIGNAL_ADD) return SHMEMG_ERR_ARG;
            if (!shmemg_in_range(w, o.sig_off, 8)) return SHMEMG_ERR_RANGE;
            if (o.sig_off & 7) return SHMEMG_ERR_ALIGN;
        }
        return SHMEMG_OK;
    }
    // AMOs
    if (!shmemg_in_range(w, o.rem_off, 8)) return SHMEMG_ERR_RANGE;
    if (o.rem_off & 7) return SHMEMG_ERR_ALIGN;
    if (o.opcode != SHMEMG_OP_ATOMIC_ADD) {
        if (!shmemg_in_range(w, o.loc_off, 8)) return SHMEMG_ERR_RANGE;
        if (o.loc_off & 7) return SHMEMG_ERR_ALIGN;
    }
    return SHMEMG_OK;
}

static bool is_marker(uint8_t opc) {
    return opc == SHMEMG_OP_FENCE || opc == SHMEMG_OP_QUIET || opc == SHMEMG_OP_BARRIER_ALL;
}
static bool is_amo(uint8_t opc) { return opc >= SHMEMG_OP_ATOMIC_ADD && opc <= SHMEMG_OP_ATOMIC_COMPARE_SWAP; }

static uint32_t pick_tile_bytes(const shmemg_world *w, const shmemg_op_t *ops, size_t nops) {
    if (w->tile_bytes_override) return (uint32_t)w->tile_bytes_override;
    uint64_t total = 0;
    for (size_t i = 0; i < nops; ++i)
        if (ops[i].opcode >= SHMEMG_OP_PUT && ops[i].opcode <= SHMEMG_OP_PUT_SIGNAL) total += ops[i].nbytes;
    const uint64_t grid = (uint64_t)w->sm_count * w->ctas_per_sm;
    uint64_t want = total / (grid * 8) + 1;            // aim at >= 8 tiles per resident CTA
    uint32_t tb = 8192;
    while (tb < want && tb < 65536) tb <<= 1;
    return tb;
}

struct PlanSizes { size_t real_ops, ntiles, total; size_t ops_off, tiles_off, done_off, arrive_off; uint32_t tile_bytes; };

static PlanSizes plan_sizes(const shmemg_world *w, const shmemg_op_t *ops, size_t nops) {
    PlanSizes s{};
    s.tile_bytes = pick_tile_bytes(w, ops, nops);
    size_t run = 0;
    for (size_t i = 0; i < nops; ++i) {
        const uint8_t opc = ops[i].opcode;
        if (is_marker(opc)) { run = 0; continue; }
        s.real_ops++;
        if (is_amo(opc)) {
            if (run == 0 || run == AMO_RUN_MAX) { s.ntiles++; run = 0; }
            run++;
            continue;
        }
        run = 0;
        if (opc == SHMEMG_OP_SIGNAL_WAIT_UNTIL) s.ntiles++;
        else s.ntiles += ops[i].nbytes <= s.tile_bytes ? 1 : (ops[i].nbytes + s.tile_bytes - 1) / s.tile_bytes;
    }
    auto up = [](size_t x) { return (x + 255) / 256 * 256; };
    s.ops_off = sizeof(PlanHeader);
    s.tiles_off = s.ops_off + up(s.real_ops * sizeof(DevOp));
    s.done_off = s.tiles_off + up(s.ntiles * sizeof(Tile));
    s.arrive_off = s.done_off + up(((size_t)w->npes + 1) * 4);
    s.total = s.arrive_off + up(s.real_ops * 4) + 256;
    return s;
}

extern "C" size_t shmemg_batch_plan_bytes(const shmemg_world_t *w, const shmemg_op_t *ops_host, size_t nops) {
    if (!w || (!ops_host && nops)) return 0;
    return plan_sizes(w, ops_host, nops).total;
}

extern "C" int shmemg_batch_create(shmemg_world_t *w, const shmemg_op_t *ops, size_t nops, void *plan_dev,
                                   size_t plan_bytes, void *stream, shmemg_batch_t **out, size_t *bad_index) {
    if (!w || !out || !plan_dev || (!ops && nops)) return SHMEMG_ERR_ARG;
    *out = nullptr;
    if ((uintptr_t)plan_dev % 256) return SHMEMG_ERR_ALIGN;
    for (size_t i = 0; i < nops; ++i) {
        int rc = validate_op(w, ops[i]);
        if (rc) {
            if (bad_index) *bad_index = i;
            return rc;
        }
    }
    const PlanSizes ps = plan_sizes(w, ops, nops);
    if (plan_bytes < ps.total) return SHMEMG_ERR_NOMEM;
    if (ps.ntiles >= 0xffffffffull || ps.real_ops >= 0xffffffffull) return SHMEMG_ERR_NOMEM;

    std::vector<uint8_t> host(ps.total, 0);
    PlanHeader *hdr = reinterpret_cast<PlanHeader *>(host.data());
    DevOp *dops = reinterpret_cast<DevOp *>(host.data() + ps.ops_off);
    Tile *tiles = reinterpret_cast<Tile *>(host.data() + ps.tiles_off);
    hdr->ntiles = (uint32_t)ps.ntiles;
    hdr->nops = (uint32_t)ps.real_ops;
    hdr->npes = (uint32_t)w->npes;
    hdr->tile_bytes = ps.tile_bytes;
    hdr->ops_off = ps.ops_off; hdr->tiles_off = ps.tiles_off; hdr->done_off = ps.done_off; hdr->arrive_off = ps.arrive_off;

    // forward pass: dependencies.  issued[p] = real ops of PE p so far; thresh[p] = what p's next op must see.
    std::vector<uint32_t> issued(w->npes, 0), thresh(w->npes, 0);
    std::vector<uint32_t> src_index;            // real op -> index in the caller's array
    src_index.reserve(ps.real_ops);
    uint32_t all_issued = 0, all_thresh = 0;
    size_t k = 0, nt = 0, run = 0;
    for (size_t i = 0; i < nops; ++i) {
        const shmemg_op_t &o = ops[i];
        if (o.opcode == SHMEMG_OP_FENCE || o.opcode == SHMEMG_OP_QUIET) {
            thresh[o.initiator_pe] = issued[o.initiator_pe]; run = 0; continue;
        }
        if (o.opcode == SHMEMG_OP_BARRIER_ALL) { all_thresh = all_issued; run = 0; continue; }
        DevOp &d = dops[k];
        const int ini = o.initiator_pe;
        d.kind = o.opcode;
        d.initiator = (uint32_t)ini;
        d.dep_pe = thresh[ini];
        d.dep_all = all_thresh;
        d.value = o.value;
        d.cond = o.cond;
        d.nbytes = o.nbytes;
        if (o.opcode == SHMEMG_OP_PUT || o.opcode == SHMEMG_OP_PUT_SIGNAL) {
            d.dst = (uint64_t)shmemg_addr(w, o.target_pe, o.rem_off);
            d.src = (uint64_t)shmemg_addr(w, ini, o.loc_off);
            if (o.opcode == SHMEMG_OP_PUT_SIGNAL) {
                d.sig = (uint64_t)shmemg_addr(w, o.target_pe, o.sig_off);
                d.kind |= (uint32_t)o.sig_op << 8;
            }
        } else if (o.opcode == SHMEMG_OP_GET) {
            d.dst = (uint64_t)shmemg_addr(w, ini, o.loc_off);
            d.src = (uint64_t)shmemg_addr(w, o.target_pe, o.rem_off);
        } else if (o.opcode == SHMEMG_OP_SIGNAL_WAIT_UNTIL) {
            d.sig = (uint64_t)shmemg_addr(w, ini, o.loc_off);
            d.kind |= (uint32_t)o.cmp << 8;
        } else {   // AMO
            d.dst = (uint64_t)shmemg_addr(w, o.target_pe, o.rem_off);
            d.src = o.opcode == SHMEMG_OP_ATOMIC_ADD ? 0 : (uint64_t)shmemg_addr(w, ini, o.loc_off);
            d.nbytes = 8;
        }
        // tiles
        if (is_amo(o.opcode)) {
            if (run == 0 || run == AMO_RUN_MAX) { tiles[nt].op = (uint32_t)k; tiles[nt].sub = 0; nt++; run = 0; }
            tiles[nt - 1].sub++;
            run++;
        } else {
            run = 0;
            const size_t n = (o.opcode == SHMEMG_OP_SIGNAL_WAIT_UNTIL || o.nbytes <= ps.tile_bytes)
                                 ? 1 : (o.nbytes + ps.tile_bytes - 1) / ps.tile_bytes;
            for (size_t s = 0; s < n; ++s) { tiles[nt].op = (uint32_t)k; tiles[nt].sub = (uint32_t)s; nt++; }
        }
        issued[ini]++; all_issued++;
        if (o.opcode == SHMEMG_OP_SIGNAL_WAIT_UNTIL) thresh[ini] = issued[ini];   // later ops of this PE follow the wait
        src_index.push_back((uint32_t)i);
        k++;
    }
    // backward pass: which ops does a later marker depend on?
    {
        std::vector<uint8_t> later_pe(w->npes, 0);
        bool later_all = false;
        size_t kk = ps.real_ops;
        for (size_t i = nops; i-- > 0;) {
            const shmemg_op_t &o = ops[i];
            if (o.opcode == SHMEMG_OP_FENCE || o.opcode == SHMEMG_OP_QUIET) { later_pe[o.initiator_pe] = 1; continue; }
            if (o.opcode == SHMEMG_OP_BARRIER_ALL) { later_all = true; continue; }
            kk--;
            // A wait makes the PE's LATER ops depend on done[p] reaching the wait's own count, so the wait and
            // every earlier op of that PE must be counted.
            if (o.opcode == SHMEMG_OP_SIGNAL_WAIT_UNTIL) later_pe[o.initiator_pe] = 1;
            if (later_pe[o.initiator_pe]) dops[kk].kind |= OPF_COUNT_PE;
            if (later_all) dops[kk].kind |= OPF_COUNT_ALL;
        }
    }

    cudaStream_t st = (cudaStream_t)stream;
    SHMEMG_CUDA(w, cudaMemcpyAsync(plan_dev, host.data(), ps.total, cudaMemcpyHostToDevice, st));
    SHMEMG_CUDA(w, cudaStreamSynchronize(st));

    shmemg_batch *b = new shmemg_batch();
    b->w = w;
    b->plan_dev = (uint8_t *)plan_dev;
    b->ntiles = (uint32_t)ps.ntiles;
    const uint64_t maxgrid = (uint64_t)w->sm_count * w->ctas_per_sm;
    b->grid = (uint32_t)(ps.ntiles < maxgrid ? (ps.ntiles ? ps.ntiles : 1) : maxgrid);
    *out = b;
    return SHMEMG_OK;
}

extern "C" int shmemg_batch_destroy(shmemg_batch_t *b) {
    if (!b) return SHMEMG_ERR_ARG;
    delete b;
    return SHMEMG_OK;
}
extern "C" int shmemg_batch_launches(const shmemg_batch_t *b) { return b ? (b->ntiles ? 1 : 0) : SHMEMG_ERR_ARG; }

extern "C" int shmemg_batch_enqueue_on_stream(shmemg_world_t *w, shmemg_batch_t *b, void *stream) {
    if (!w || !b || b->w != w) return SHMEMG_ERR_ARG;
    if (b->ntiles == 0) return SHMEMG_OK;
    k_batch_exec<<<b->grid, SHMEMG_THREADS, 0, (cudaStream_t)stream>>>(b->plan_dev);
    SHMEMG_CUDA(w, cudaGetLastError());
    return SHMEMG_OK;
}

// ---------------------------------------------------------------------------------------------------------
// single operations on a stream
// ---------------------------------------------------------------------------------------------------------
static int launch_copy(shmemg_world *w, uint8_t *dst, const uint8_t *src, size_t nbytes, unsigned long long *sig,
                       uint64_t sig_value, int sig_op, cudaStream_t st) {
    if (nbytes == 0 && !sig) return SHMEMG_OK;
    const uint64_t maxgrid = (uint64_t)w->sm_count * w->ctas_per_sm;
    uint32_t tb = 8192;
    while (tb < 65536 && nbytes / tb > maxgrid * 8) tb <<= 1;
    if (w->tile_bytes_override) tb = (uint32_t)w->tile_bytes_override;
    uint64_t ntiles = (nbytes + tb - 1) / tb;
    uint32_t grid = (uint32_t)(ntiles < maxgrid ? (ntiles ? ntiles : 1) : maxgrid);
    unsigned *counter = sig ? &w->ctl->sig_counter[(w->sig_seq++) % SHMEMG_SIG_SLOTS] : nullptr;
    k_copy_single<<<grid, SHMEMG_THREADS, 0, st>>>(dst, src, nbytes, tb, sig, sig_value, sig_op, counter);
    SHMEMG_CUDA(w, cudaGetLastError());
    return SHMEMG_OK;
}

extern "C" int shmemg_put_on_stream(shmemg_world_t *w, uint64_t dest_off, uint64_t source_off, size_t nbytes, int pe,
                                    int target_pe, void *stream) {
    if (!w) return SHMEMG_ERR_ARG;
    if (!shmemg_pe_ok(w, pe) || !shmemg_pe_ok(w, target_pe)) return SHMEMG_ERR_PE;
    if (!shmemg_in_range(w, dest_off, nbytes) || !shmemg_in_range(w, source_off, nbytes)) return SHMEMG_ERR_RANGE;
    return launch_copy(w, shmemg_addr(w, target_pe, dest_off), shmemg_addr(w, pe, source_off), nbytes, nullptr, 0, 0,
                       (cudaStream_t)stream);
}
extern "C" int shmemg_get_on_stream(shmemg_world_t *w, uint64_t dest_off, uint64_t source_off, size_t nbytes, int pe,
                                    int target_pe, void *stream) {
    if (!w) return SHMEMG_ERR_ARG;
    if (!shmemg_pe_ok(w, pe) || !shmemg_pe_ok(w, target_pe)) return SHMEMG_ERR_PE;
    if (!shmemg_in_range(w, dest_off, nbytes) || !shmemg_in_range(w, source_off, nbytes)) return SHMEMG_ERR_RANGE;
    return launch_copy(w, shmemg_addr(w, pe, dest_off), shmemg_addr(w, target_pe, source_off), nbytes, nullptr, 0, 0,
                       (cudaStream_t)stream);
}
extern "C" int shmemg_put_signal_on_stream(shmemg_world_t *w, uint64_t dest_off, uint64_t source_off, size_t nbytes,
                                           uint64_t sig_off, uint64_t signal, int sig_op, int pe, int target_pe,
                                           void *stream) {
    if (!w || sig_op < SHMEMG_SIGNAL_SET || sig_op > SHMEMG_SIGNAL_ADD) return SHMEMG_ERR_ARG;
    if (!shmemg_pe_ok(w, pe) || !shmemg_pe_ok(w, target_pe)) return SHMEMG_ERR_PE;
    if (!shmemg_in_range(w, dest_off, nbytes) || !shmemg_in_range(w, source_off, nbytes) ||
        !shmemg_in_range(w, sig_off, 8))
        return SHMEMG_ERR_RANGE;
    if (sig_off & 7) return SHMEMG_ERR_ALIGN;
    return launch_copy(w, shmemg_addr(w, target_pe, dest_off), shmemg_addr(w, pe, source_off), nbytes,
                       (unsigned long long *)shmemg_addr(w, target_pe, sig_off), signal, sig_op, (cudaStream_t)stream);
}
extern "C" int shmemg_signal_wait_until_on_stream(shmemg_world_t *w, uint64_t sig_off, int cmp, uint64_t value, int pe,
                                                  void *stream) {
    if (!w || cmp < SHMEMG_CMP_EQ || cmp > SHMEMG_CMP_LE) return SHMEMG_ERR_ARG;
    if (!shmemg_pe_ok(w, pe)) return SHMEMG_ERR_PE;
    if (!shmemg_in_range(w, sig_off, 8)) return SHMEMG_ERR_RANGE;
    if (sig_off & 7) return SHMEMG_ERR_ALIGN;
    k_wait_until<<<1, 1, 0, (cudaStream_t)stream>>>((const unsigned long long *)shmemg_addr(w, pe, sig_off), cmp, value);
    SHMEMG_CUDA(w, cudaGetLastError());
    return SHMEMG_OK;
}
extern "C" int shmemg_fence_on_stream(shmemg_world_t *w, int pe, void *stream) {
    (void)stream;
    if (!w) return SHMEMG_ERR_ARG;
    return shmemg_pe_ok(w, pe) ? SHMEMG_OK : SHMEMG_ERR_PE;
}
extern "C" int shmemg_quiet_on_stream(shmemg_world_t *w, int pe, void *stream) {
    return shmemg_fence_on_stream(w, pe, stream);
}
extern "C" int shmemg_quiet(shmemg_world_t *w, int pe, void *stream) {
    int rc = shmemg_fence_on_stream(w, pe, stream);
    if (rc) return rc;
    SHMEMG_CUDA(w, cudaStreamSynchronize((cudaStream_t)stream));
    return SHMEMG_OK;
}
