/*
 * shmemg_probe.h -- CEILING PROBES used by bench.py to measure, on the same box and in the same run,
 * the denominators the AMO paths are reported against (SURVEY.md 8(d) "L2-atomic ceiling").
 *
 * NOT operations of the specification: a probe issues the bare L2 atomic instruction of an AMO path
 * (red.global.add.u64 / atom.global.add.u64 / atom.global.cas.b64) at addresses it derives from a hash
 * of the op index, with no descriptor reads and no fetched-value writes, so its rate is what the L2
 * atomic units sustain for that address distribution.  Same conventions as shmemg.h.
 */
#ifndef SHMEMG_PROBE_H
#define SHMEMG_PROBE_H
#include "shmemg.h"
#ifdef __cplusplus
extern "C" {
#endif

enum { SHMEMG_PROBE_RED_ADD = 0, SHMEMG_PROBE_ATOM_ADD = 1, SHMEMG_PROBE_ATOM_CAS = 2 };

/* Issue `n` atomics on `stream`: op i targets u64 heap[pe(i)][sym_off + 8*wd(i)] with pe(i), wd(i) derived from a
 * 64-bit hash of i by multiply-high (uniformly random over npes*words_per_pe words, no integer division), adding 0 (RED_ADD / ATOM_ADD) or comparing against a value the
 * word never holds (ATOM_CAS), so the heap is left unchanged.  words_per_pe >= 1; the object at sym_off must hold
 * 8*words_per_pe bytes.  Fetched values are xor-reduced per thread and stored only if the reduction is a value it
 * cannot take (keeps the atom.* results live without output traffic). */
SHMEMG_API int shmemg_probe_atomic_on_stream(shmemg_world_t *w, int mode, uint64_t sym_off, uint64_t words_per_pe,
                                             size_t n, void *stream);

/* The same bare atomics on a GIVEN address stream: op i targets u64 heap[tgt_pe[i]][sym_off + 8*elem_idx[i]] (DEVICE arrays of n
 * entries: the workload's own operand arrays, e.g. the RMAT endpoints of config C4), or, with tgt_pe == elem_idx == NULL, on the
 * ONE word heap[0][sym_off].  aggregate != 0: a warp issues one atomic per distinct address (what SHMEMG_AMO_WARP_AGGREGATE
 * does).  Adds 0 / compares against a value the word never holds: the heap is left unchanged.  These are the like-for-like
 * ceilings of SURVEY.md 8(d) (iii) "RMAT-skewed as C4" and (iv) "single address". */
SHMEMG_API int shmemg_probe_atomic_stream_on_stream(shmemg_world_t *w, int mode, uint64_t sym_off, const int32_t *tgt_pe,
                                                    const uint32_t *elem_idx, size_t n, int aggregate, void *stream);

/* Plain device copy ceiling with the library's own streaming loop: heap[pe_dst][dst_off..] = heap[pe_src][src_off..]
 * is shmemg_put_on_stream; this probe instead reports nothing new and exists only so bench.py can time the kernel
 * on one contiguous `nbytes` range per PE pair for every PE at once (npes independent copies, one launch). */
SHMEMG_API int shmemg_probe_copy_all_on_stream(shmemg_world_t *w, uint64_t dst_off, uint64_t src_off, size_t nbytes,
                                               void *stream);

#ifdef __cplusplus
}
#endif
#endif
