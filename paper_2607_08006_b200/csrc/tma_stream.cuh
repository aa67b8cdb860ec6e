// tma_stream.cuh -- bulk-copy (TMA) streaming pipelines shared by the copy-class kernels (sm_100a).
//
// One thread per CTA drives a ring of SHMEMG_TMA_STAGES shared-memory stages of SHMEMG_TMA_TILE bytes:
//   load  : cp.async.bulk global -> shared, completion counted on an mbarrier        (SASS UBLKCP.S.G)
//   store : cp.async.bulk shared -> global, completion tracked by bulk async-groups   (SASS UBLKCP.G.S)
// STAGES-1 loads are kept in flight ahead of the store front, so about 96 KiB per SM is outstanding towards HBM with
// no registers and a single issuing thread.  Requirements: 16-byte aligned source, destination and size; callers
// fall back to the register path (copy_coop) otherwise.
#pragma once
#include "internal.cuh"

#define SHMEMG_TMA_SMEM ((size_t)SHMEMG_TMA_STAGES * SHMEMG_TMA_TILE)

// FnItem(k, src, dst, n): the k-th work item of the launch (n <= SHMEMG_TMA_TILE, all 16-byte aligned).
// Items first, first+step, ... < nitems are copied by the calling thread; returns after every store has completed.
template <typename FnItem>
__device__ __forceinline__ void tma_stream_copy(uint8_t *stage, uint64_t *full, size_t first, size_t step, size_t nitems,
                                                FnItem item) {
    const size_t mine = first < nitems ? (nitems - first + step - 1) / step : 0;
    auto issue_load = [&](size_t it) {
        const uint8_t *s; uint8_t *d; unsigned n;
        item(first + it * step, s, d, n);
        const int st = (int)(it % SHMEMG_TMA_STAGES);
        mbar_arrive_expect_tx(&full[st], n);
        bulk_g2s(stage + (size_t)st * SHMEMG_TMA_TILE, s, n, &full[st]);
    };
    for (size_t it = 0; it < mine && it < SHMEMG_TMA_STAGES - 1; ++it) issue_load(it);
    for (size_t it = 0; it < mine; ++it) {
        const int st = (int)(it % SHMEMG_TMA_STAGES);
        mbar_wait(&full[st], (unsigned)((it / SHMEMG_TMA_STAGES) & 1));
        const uint8_t *s; uint8_t *d; unsigned n;
        item(first + it * step, s, d, n);
        bulk_s2g(d, stage + (size_t)st * SHMEMG_TMA_TILE, n);
        bulk_commit();
        if (it + SHMEMG_TMA_STAGES - 1 < mine) {
            bulk_wait_read<1>();              // the store issued one iteration ago no longer reads its stage
            issue_load(it + SHMEMG_TMA_STAGES - 1);
        }
    }
    bulk_wait<0>();
}

__device__ __forceinline__ void tma_stream_init(uint64_t *full) {
    for (int s = 0; s < SHMEMG_TMA_STAGES; ++s) mbar_init(&full[s], 1);
    mbar_init_fence();
}
