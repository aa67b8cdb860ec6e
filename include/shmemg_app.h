/*
 * shmemg_app.h -- APPLICATION-side kernels of the halo-exchange workload (BASELINE config 2).
 *
 * NOT part of the specification's operations: this is the stencil application's own compute
 * (perturb the interior, pack faces, checksum what was received; SURVEY.md readings 21-23), kept in
 * the library only so the tests and bench.py can drive the workload on the GPU.  It is excluded from
 * the timed library path.  Same conventions as shmemg.h (symmetric offsets, raw stream as void *).
 */
#ifndef SHMEMG_APP_H
#define SHMEMG_APP_H
#include "shmemg.h"
#ifdef __cplusplus
extern "C" {
#endif

/* For all 8 PEs of a 2x2x2 world (PE p = (px*2+py)*2+pz): U[c] += (mix64(seed, round, g(c)) & 0xFFFF) * 2^-30
 * where U is a B^3 fp64 block at U_off (x-major) and g(c) is c's index in the (2B)^3 global grid. */
SHMEMG_API int shmemg_app_halo_perturb_on_stream(shmemg_world_t *w, uint64_t U_off, uint32_t B, uint64_t seed,
                                                 uint64_t round, void *stream);
/* For all 8 PEs and all 6 faces f = 2*axis+dir: send[f][a*B+b] = boundary plane of U (dir 0: index 0,
 * dir 1: index B-1 along axis; remaining axes in order). */
SHMEMG_API int shmemg_app_halo_pack_on_stream(shmemg_world_t *w, uint64_t send_off, uint64_t U_off, uint32_t B,
                                              void *stream);
/* out[p*nseg + s] = sum_k u64(heap[p][sym_off + s*seg_bytes + 8k]) * (2k+1) mod 2^64, k < seg_bytes/8.
 * `out` is a DEVICE array of npes*nseg uint64, overwritten. */
SHMEMG_API int shmemg_app_checksum64_on_stream(shmemg_world_t *w, uint64_t *out, uint64_t sym_off, uint64_t seg_bytes,
                                               uint32_t nseg, void *stream);
/* The halo application DEVICE-INITIATED and persistent ("kernel-boundary
 * synchronisation limits strong scaling"): ONE cooperative kernel runs rounds first_round .. first_round+rounds-1.  Every PE is
 * a group of thread blocks.  Six "face blocks" per PE: perturb the boundary cells, synchronise among themselves, put one face
 * each straight out of the cube (shmemg_dev_ibput_block) into the neighbour's ghost[round & 1][face'], signal sig[face'] =
 * round (shmemg_dev_signal_block) and wait for their own incoming face (shmemg_dev_signal_wait_until_block).  All other
 * blocks perturb the interior and never wait inside a round; before the next round they check that the round's six faces
 * have arrived.  No send buffer, no pack kernel, no kernel boundary between rounds; the exchange is hidden behind the interior
 * update.  Results (U, ghost, sig) are bit-identical to rounds of perturb + pack + put_signal/wait batches.
 * Returns SHMEMG_ERR_NOMEM if the blocks cannot all be co-resident.  B <= 1024. */
SHMEMG_API int shmemg_app_halo_persistent_on_stream(shmemg_world_t *w, uint64_t U_off, uint64_t ghost_off, uint64_t sig_off,
                                                    uint32_t B, uint64_t seed, uint64_t first_round, uint32_t rounds,
                                                    void *stream);
#ifdef __cplusplus
}
#endif
#endif
