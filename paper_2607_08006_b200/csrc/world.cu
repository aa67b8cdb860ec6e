// world.cu -- lifecycle, capability query, symmetric-heap allocator, PE->address translation.
// Host-only bookkeeping; the only device work is memset / memcpy.
#include <stdlib.h>
#include <string.h>

#include "internal.cuh"

static size_t round_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

// SHMEMG_SYMMETRIC_SIZE: bytes with optional K/M/G suffix (heap traits via environment)
static size_t env_heap_bytes() {
    const char *s = getenv("SHMEMG_SYMMETRIC_SIZE");
    if (!s || !*s) return 0;
    char *end = nullptr;
    double v = strtod(s, &end);
    if (v <= 0) return 0;
    size_t mul = 1;
    if (end && *end) {
        switch (*end) {
        case 'k': case 'K': mul = 1ull << 10; break;
        case 'm': case 'M': mul = 1ull << 20; break;
        case 'g': case 'G': mul = 1ull << 30; break;
        default: return 0;
        }
    }
    return (size_t)(v * (double)mul);
}

extern "C" size_t shmemg_slab_bytes_required(int npes, size_t heap_bytes_per_pe) {
    if (npes < 1) return 0;
    if (heap_bytes_per_pe == 0) heap_bytes_per_pe = env_heap_bytes();
    if (heap_bytes_per_pe == 0) return 0;
    return (size_t)npes * round_up(heap_bytes_per_pe, SHMEMG_STRIDE_ALIGN) + SHMEMG_CTL_BYTES + SHMEMG_ARENA_BYTES;
}

extern "C" int shmemg_init(int npes, size_t heap_bytes_per_pe, void *device_slab, size_t slab_bytes,
                           shmemg_world_t **out) {
    if (!out) return SHMEMG_ERR_ARG;
    *out = nullptr;
    if (npes < 1 || !device_slab) return SHMEMG_ERR_ARG;
    if (heap_bytes_per_pe == 0) heap_bytes_per_pe = env_heap_bytes();
    if (heap_bytes_per_pe == 0) return SHMEMG_ERR_ARG;
    if ((uintptr_t)device_slab % SHMEMG_STRIDE_ALIGN) return SHMEMG_ERR_ALIGN;
    const size_t need = shmemg_slab_bytes_required(npes, heap_bytes_per_pe);
    if (slab_bytes < need) return SHMEMG_ERR_NOMEM;

    cudaPointerAttributes attr;
    if (cudaPointerGetAttributes(&attr, device_slab) != cudaSuccess || attr.type != cudaMemoryTypeDevice) {
        cudaGetLastError();
        return SHMEMG_ERR_ARG;     // managed/unified/host memory is outside the baseline model
    }
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, attr.device) != cudaSuccess) return SHMEMG_ERR_CUDA;
    if (prop.major != 10) return SHMEMG_ERR_NODEVICE;   // sm_100a cubins only: fail loudly elsewhere
    int cur = -1;
    cudaGetDevice(&cur);
    if (cur != attr.device && cudaSetDevice(attr.device) != cudaSuccess) return SHMEMG_ERR_CUDA;

    shmemg_world *w = new shmemg_world();
    w->npes = npes;
    w->device = attr.device;
    w->sm_count = prop.multiProcessorCount;
    w->heap_bytes = heap_bytes_per_pe;
    w->stride = round_up(heap_bytes_per_pe, SHMEMG_STRIDE_ALIGN);
    w->base = (uint8_t *)device_slab;
    w->slab_bytes = slab_bytes;
    w->ctl = (CtlRegion *)(w->base + (size_t)npes * w->stride);
    w->arena = (uint8_t *)w->ctl + SHMEMG_CTL_BYTES;
    w->free_list[0] = heap_bytes_per_pe;
#ifdef SHMEMG_EXPERIMENTS                                               // tuning knobs: not in the shipped build (_build.py sets no such flag)
    if (const char *s = getenv("SHMEMG_CTAS_PER_SM")) {
        int v = atoi(s);
        if (v >= 1 && v <= 8) w->ctas_per_sm = v;
    }
    if (const char *s = getenv("SHMEMG_TILE_BYTES")) {
        long v = atol(s);
        if (v >= 1024) w->tile_bytes_override = (size_t)v;
    }
#endif
    if (getenv("SHMEMG_NO_PDL")) w->dependent_launch = false;       // read once, here; shmemg_set_dependent_launch changes it later
    static_assert(sizeof(CtlRegion) <= SHMEMG_CTL_BYTES, "control region too small");
    cudaError_t e = cudaMemset(w->ctl, 0, SHMEMG_CTL_BYTES);
    if (e == cudaSuccess) e = cudaDeviceSynchronize();
    if (e != cudaSuccess) {
        delete w;
        return SHMEMG_ERR_CUDA;
    }
    *out = w;
    return SHMEMG_OK;
}

extern "C" int shmemg_finalize(shmemg_world_t *w) {
    if (!w) return SHMEMG_ERR_ARG;
    shmemg_shard_release(w);
    delete w;
    return SHMEMG_OK;
}

extern "C" int shmemg_n_pes(const shmemg_world_t *w) { return w ? w->npes : SHMEMG_ERR_ARG; }
extern "C" size_t shmemg_heap_bytes(const shmemg_world_t *w) { return w ? w->heap_bytes : 0; }
extern "C" size_t shmemg_heap_stride(const shmemg_world_t *w) { return w ? w->stride : 0; }
extern "C" const char *shmemg_last_cuda_error(const shmemg_world_t *w) { return w ? w->last_cuda_error.c_str() : ""; }

extern "C" int shmem_query_capabilities(const shmemg_world_t *w, int team, uint64_t *caps) {
    if (!w || !caps) return SHMEMG_ERR_ARG;
    if (team >= SHMEMG_TEAM_USER0 && (size_t)(team - SHMEMG_TEAM_USER0) < w->teams.size()) team = SHMEM_TEAM_WORLD;
    if (team != SHMEM_TEAM_WORLD && team != SHMEM_DEVICE_TEAM_WORLD && team != SHMEM_DEVICE_TEAM_SHARED)
        return SHMEMG_ERR_ARG;
    // Capabilities are per team.  All PEs share one GPU, so the three predefined teams have
    // the same membership; they differ in which initiation paths they scope (L357, L412).
    uint64_t c = SHMEMG_CAP_GPU_HEAP_PRESENT | SHMEMG_CAP_DEFAULT_HEAP_IS_GPU | SHMEMG_CAP_PTR_DEVICE_ACCESSIBLE |
                 SHMEMG_CAP_PROGRESS_GPU_ONLY | SHMEMG_CAP_PATH_DIRECT | SHMEMG_CAP_ATOMICS_64;
    if (w->cpu_base) c |= SHMEMG_CAP_CPU_HEAP_PRESENT;      // the CPU half of the two-space model is attached (L313-L317)
    if (w->nshards > 1) c |= SHMEMG_CAP_PEER_SHARDS;        // one shard of a multi-GPU world over a load-store fabric (L194)
    if (team == SHMEM_TEAM_WORLD)
        c |= SHMEMG_CAP_HOST_INITIATED_GPU_BUFFERS | SHMEMG_CAP_STREAM_TRIGGERED | SHMEMG_CAP_STREAM_COLLECTIVES;
    else
        c |= SHMEMG_CAP_DEVICE_INITIATED | SHMEMG_CAP_DEVICE_BARRIER | SHMEMG_CAP_DEVICE_COLLECTIVES |
             SHMEMG_CAP_EXPLICIT_DEVICE_CTX;   // include/shmemg_device.cuh
    *caps = c;
    return SHMEMG_OK;
}

// ---- symmetric allocator: first fit over a coalescing free list; one offset for all PEs (a2) ---------------
static int alloc_in(std::map<uint64_t, size_t> &free_list, std::map<uint64_t, size_t> &live, size_t alignment, size_t bytes,
                    uint64_t *sym_off);
static int alloc_impl(shmemg_world *w, size_t alignment, size_t bytes, uint64_t *sym_off) {
    if (!w || !sym_off) return SHMEMG_ERR_ARG;
    return alloc_in(w->free_list, w->live, alignment, bytes, sym_off);
}
static int alloc_in(std::map<uint64_t, size_t> &free_list, std::map<uint64_t, size_t> &live, size_t alignment, size_t bytes,
                    uint64_t *sym_off) {
    if (alignment < SHMEMG_MIN_ALIGN) alignment = SHMEMG_MIN_ALIGN;
    if (alignment & (alignment - 1)) return SHMEMG_ERR_ARG;
    if (bytes == 0) bytes = 1;
    bytes = round_up(bytes, SHMEMG_MIN_ALIGN);
    for (auto it = free_list.begin(); it != free_list.end(); ++it) {
        const uint64_t start = it->first, size = it->second;
        const uint64_t a = round_up(start, alignment);
        if (a + bytes > start + size || a + bytes < a) continue;
        free_list.erase(it);
        if (a > start) free_list[start] = a - start;
        if (a + bytes < start + size) free_list[a + bytes] = start + size - (a + bytes);
        live[a] = bytes;
        *sym_off = a;
        return SHMEMG_OK;
    }
    return SHMEMG_ERR_NOMEM;
}

extern "C" int shmemg_malloc(shmemg_world_t *w, size_t bytes, uint64_t *sym_off) {
    return alloc_impl(w, SHMEMG_MIN_ALIGN, bytes, sym_off);
}
extern "C" int shmemg_align(shmemg_world_t *w, size_t alignment, size_t bytes, uint64_t *sym_off) {
    return alloc_impl(w, alignment, bytes, sym_off);
}
extern "C" int shmemg_calloc(shmemg_world_t *w, size_t count, size_t size, uint64_t *sym_off, void *stream) {
    if (size && count > SIZE_MAX / size) return SHMEMG_ERR_NOMEM;
    int rc = alloc_impl(w, SHMEMG_MIN_ALIGN, count * size, sym_off);
    if (rc) return rc;
    // zero the object in every PE's window: one strided 2-D memset
    const size_t bytes = w->live[*sym_off];
    const size_t width = (*sym_off + bytes <= w->heap_bytes) ? bytes : w->heap_bytes - *sym_off;
    SHMEMG_CUDA(w, cudaMemset2DAsync(w->base + *sym_off, w->stride, 0, width, (size_t)w->npes, (cudaStream_t)stream));
    return SHMEMG_OK;
}
static int free_in(std::map<uint64_t, size_t> &free_list, std::map<uint64_t, size_t> &live, uint64_t sym_off) {
    auto it = live.find(sym_off);
    if (it == live.end()) return SHMEMG_ERR_ARG;
    uint64_t start = it->first, size = it->second;
    live.erase(it);
    auto nxt = free_list.lower_bound(start);
    if (nxt != free_list.end() && start + size == nxt->first) {   // merge with the following block
        size += nxt->second;
        nxt = free_list.erase(nxt);
    }
    if (nxt != free_list.begin()) {                                // merge with the preceding block
        auto prv = std::prev(nxt);
        if (prv->first + prv->second == start) {
            prv->second += size;
            return SHMEMG_OK;
        }
    }
    free_list[start] = size;
    return SHMEMG_OK;
}
extern "C" int shmemg_free(shmemg_world_t *w, uint64_t sym_off) {
    if (!w) return SHMEMG_ERR_ARG;
    return free_in(w->free_list, w->live, sym_off);
}

// ---- the CPU space of the two-space model (Fig. 4) -----------------------------------------------------------
extern "C" int shmemg_cpu_heap_attach(shmemg_world_t *w, void *host_slab, size_t heap_bytes_per_pe, size_t slab_bytes) {
    if (!w || !host_slab || heap_bytes_per_pe == 0 || w->cpu_base) return SHMEMG_ERR_ARG;
    if ((uintptr_t)host_slab % SHMEMG_MIN_ALIGN) return SHMEMG_ERR_ALIGN;
    const size_t stride = round_up(heap_bytes_per_pe, SHMEMG_STRIDE_ALIGN);
    if (slab_bytes < (size_t)w->npes * stride) return SHMEMG_ERR_NOMEM;
    cudaPointerAttributes attr;
    if (cudaPointerGetAttributes(&attr, host_slab) != cudaSuccess || attr.type != cudaMemoryTypeHost) {
        cudaGetLastError();
        return SHMEMG_ERR_ARG;            // pageable or device memory: the CPU space must be page-locked host memory (L456)
    }
    w->cpu_base = (uint8_t *)host_slab;
    w->cpu_heap_bytes = heap_bytes_per_pe;
    w->cpu_stride = stride;
    w->cpu_free_list.clear(); w->cpu_live.clear();
    w->cpu_free_list[0] = heap_bytes_per_pe;
    return SHMEMG_OK;
}
extern "C" int shmemg_cpu_malloc(shmemg_world_t *w, size_t bytes, uint64_t *sym_off) {
    if (!w || !sym_off || !w->cpu_base) return SHMEMG_ERR_ARG;
    return alloc_in(w->cpu_free_list, w->cpu_live, SHMEMG_MIN_ALIGN, bytes, sym_off);
}
extern "C" int shmemg_cpu_free(shmemg_world_t *w, uint64_t sym_off) {
    if (!w || !w->cpu_base) return SHMEMG_ERR_ARG;
    return free_in(w->cpu_free_list, w->cpu_live, sym_off);
}
extern "C" void *shmemg_cpu_ptr(const shmemg_world_t *w, uint64_t sym_off, int pe) {
    if (!w || !w->cpu_base || !shmemg_pe_ok(w, pe) || sym_off >= w->cpu_heap_bytes) return nullptr;
    return w->cpu_base + (size_t)pe * w->cpu_stride + sym_off;
}

// put / get between the two spaces: GPU <-> GPU runs the copy kernels, anything that touches the CPU space is a DMA transfer
extern "C" int shmemg_put_on_stream(shmemg_world_t *w, uint64_t dest_off, uint64_t source_off, size_t nbytes, int pe, int target_pe,
                                    void *stream);
static int copy_spaces(shmemg_world *w, int dst_space, int dst_pe, uint64_t dst_off, int src_space, int src_pe, uint64_t src_off,
                       size_t nbytes, void *stream) {
    if (!w || dst_space < SHMEMG_SPACE_GPU || dst_space > SHMEMG_SPACE_CPU || src_space < SHMEMG_SPACE_GPU || src_space > SHMEMG_SPACE_CPU)
        return SHMEMG_ERR_ARG;
    if ((dst_space == SHMEMG_SPACE_CPU || src_space == SHMEMG_SPACE_CPU) && !w->cpu_base) return SHMEMG_ERR_ARG;
    if (!shmemg_pe_ok(w, dst_pe) || !shmemg_pe_ok(w, src_pe)) return SHMEMG_ERR_PE;
    const uint64_t dlim = dst_space == SHMEMG_SPACE_GPU ? w->heap_bytes : w->cpu_heap_bytes;
    const uint64_t slim = src_space == SHMEMG_SPACE_GPU ? w->heap_bytes : w->cpu_heap_bytes;
    if (dst_off > dlim || nbytes > dlim - dst_off || src_off > slim || nbytes > slim - src_off) return SHMEMG_ERR_RANGE;
    if (nbytes == 0) return SHMEMG_OK;
    uint8_t *d = dst_space == SHMEMG_SPACE_GPU ? shmemg_addr(w, dst_pe, dst_off) : w->cpu_base + (size_t)dst_pe * w->cpu_stride + dst_off;
    const uint8_t *s = src_space == SHMEMG_SPACE_GPU ? shmemg_addr(w, src_pe, src_off) : w->cpu_base + (size_t)src_pe * w->cpu_stride + src_off;
    SHMEMG_CUDA(w, cudaMemcpyAsync(d, s, nbytes, cudaMemcpyDefault, (cudaStream_t)stream));
    return SHMEMG_OK;
}
extern "C" int shmemg_put_space_on_stream(shmemg_world_t *w, int dest_space, uint64_t dest_off, int source_space, uint64_t source_off,
                                          size_t nbytes, int pe, int target_pe, void *stream) {
    if (w && dest_space == SHMEMG_SPACE_GPU && source_space == SHMEMG_SPACE_GPU)
        return shmemg_put_on_stream(w, dest_off, source_off, nbytes, pe, target_pe, stream);
    return copy_spaces(w, dest_space, target_pe, dest_off, source_space, pe, source_off, nbytes, stream);
}
extern "C" int shmemg_get_on_stream(shmemg_world_t *w, uint64_t dest_off, uint64_t source_off, size_t nbytes, int pe, int target_pe,
                                    void *stream);
extern "C" int shmemg_get_space_on_stream(shmemg_world_t *w, int dest_space, uint64_t dest_off, int source_space, uint64_t source_off,
                                          size_t nbytes, int pe, int target_pe, void *stream) {
    if (w && dest_space == SHMEMG_SPACE_GPU && source_space == SHMEMG_SPACE_GPU)
        return shmemg_get_on_stream(w, dest_off, source_off, nbytes, pe, target_pe, stream);
    return copy_spaces(w, dest_space, pe, dest_off, source_space, target_pe, source_off, nbytes, stream);
}

extern "C" void *shmemg_ptr(const shmemg_world_t *w, uint64_t sym_off, int pe) {
    if (!w || !shmemg_pe_ok(w, pe) || sym_off >= w->heap_bytes) return nullptr;
    return shmemg_addr(w, pe, sym_off);
}

extern "C" int shmemg_heap_write_on_stream(shmemg_world_t *w, int pe, uint64_t dst_off, const void *src_host,
                                           size_t nbytes, void *stream) {
    if (!w || (!src_host && nbytes)) return SHMEMG_ERR_ARG;
    if (!shmemg_pe_ok(w, pe)) return SHMEMG_ERR_PE;
    if (!shmemg_in_range(w, dst_off, nbytes)) return SHMEMG_ERR_RANGE;
    if (nbytes == 0) return SHMEMG_OK;
    SHMEMG_CUDA(w, cudaMemcpyAsync(shmemg_addr(w, pe, dst_off), src_host, nbytes, cudaMemcpyHostToDevice,
                                   (cudaStream_t)stream));
    return SHMEMG_OK;
}
extern "C" int shmemg_heap_read_on_stream(shmemg_world_t *w, int pe, void *dst_host, uint64_t src_off,
                                          size_t nbytes, void *stream) {
    if (!w || (!dst_host && nbytes)) return SHMEMG_ERR_ARG;
    if (!shmemg_pe_ok(w, pe)) return SHMEMG_ERR_PE;
    if (!shmemg_in_range(w, src_off, nbytes)) return SHMEMG_ERR_RANGE;
    if (nbytes == 0) return SHMEMG_OK;
    SHMEMG_CUDA(w, cudaMemcpyAsync(dst_host, shmemg_addr(w, pe, src_off), nbytes, cudaMemcpyDeviceToHost,
                                   (cudaStream_t)stream));
    return SHMEMG_OK;
}

// Programmatic dependent launch of the batch executor and the device planner (see include/shmemg.h for when to turn it off).
extern "C" int shmemg_set_dependent_launch(shmemg_world_t *w, int enable) {
    if (!w) return SHMEMG_ERR_ARG;
    w->dependent_launch = enable != 0;
    return SHMEMG_OK;
}
