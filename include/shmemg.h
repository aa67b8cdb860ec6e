/*
 * shmemg.h -- C ABI of the B200-native GPU-aware OpenSHMEM hot path.
 *
 * What this library is: the data-parallel hot path of the "OpenSHMEM Auxiliary Specification for
 * GPU-Aware Communication" (arxiv/paper_2607_08006; cited below as PAPER L<line> of PAPER.md):
 * batched one-sided operations on a GPU-scoped symmetric heap, executed for N logical PEs whose heaps
 * are co-resident in one B200's HBM.  Every step of the path runs in hand-written sm_100a kernels;
 * there is no CPU fallback and no dependence on any other library than the CUDA runtime.
 *
 * Conventions
 *   - All N PEs live in one process, so every routine OpenSHMEM scopes to "the calling PE" takes an
 *     explicit initiator `pe`.  Argument order follows OpenSHMEM: (dest, source, nbytes, pe).
 *   - GPU-resident operands are SYMMETRIC OFFSETS (uint64_t byte offsets into every PE's heap window),
 *     never raw pointers: "GPU-resident operands MUST be allocated from a symmetric space" (PAPER L287,
 *     L351: "should not require device code to perform dynamic pointer classification").  The address of
 *     offset `off` on PE `pe` is  slab + pe*heap_stride + off  ("predictable,
 *     computable address offsets").
 *   - `stream` arguments are raw `cudaStream_t` values passed as `void *` (NULL = legacy default stream).
 *   - Pointers are marked HOST or DEVICE.  The library never allocates or frees device memory: the
 *     caller owns the slab and every DEVICE array it passes, and must keep them valid until the stream
 *     has passed the call.  The library owns only host bookkeeping plus a control region it carves from
 *     the tail of the slab -- and one fixed 8 MiB device array that is part of its image (the scratch of
 *     shmemg_atomic_fetch_add_batch_static_on_stream, for callers that cannot provide any).
 *   - Every routine returns SHMEMG_OK (0) or a negative SHMEMG_ERR_* for host-checkable misuse; nothing
 *     is enqueued on error.  Data races, overlapping unordered writes and unsatisfiable waits are
 *     undefined behaviour; an unsatisfiable wait hangs the stream (prohibited pattern,
 *     PAPER L404).
 *   - Threads: a world handle is NOT thread-safe.  Its host bookkeeping (allocator, team views, launch state) is
 *     unsynchronised, and the team collectives run the world kernels on a temporarily narrowed view of the world
 *     object: calls on ONE world from several host threads must be serialised by the caller.  Different worlds are
 *     independent.
 *   - Execution path: every `_on_stream` routine is a HOST-ISSUED,
 *     STREAM-TRIGGERED operation "whose execution is ordered relative to a GPU stream"; the library
 *     "may use internal GPU kernels to accelerate" it.  Effects are visible to later work on the same
 *     stream; host visibility needs cudaStreamSynchronize, which shmemg_quiet does.
 */
#ifndef SHMEMG_H
#define SHMEMG_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define SHMEMG_API __attribute__((visibility("default")))

typedef struct shmemg_world shmemg_world_t;   /* opaque, HOST */
typedef struct shmemg_batch shmemg_batch_t;   /* opaque, HOST: a planned op batch */

/* ---- return codes -------------------------------------------------------------------------- */
enum {
    SHMEMG_OK = 0,
    SHMEMG_ERR_ARG = -1,      /* NULL handle/pointer, bad enum, npes < 1                      */
    SHMEMG_ERR_PE = -2,       /* pe outside [0, npes)                                         */
    SHMEMG_ERR_RANGE = -3,    /* offset + size outside the heap window                        */
    SHMEMG_ERR_ALIGN = -4,    /* AMO / signal word not 8-byte aligned, typed buffer misaligned */
    SHMEMG_ERR_NOMEM = -5,    /* symmetric heap exhausted / slab or plan buffer too small     */
    SHMEMG_ERR_CUDA = -6,     /* a CUDA runtime call failed (see shmemg_last_cuda_error)       */
    SHMEMG_ERR_OVERLAP = -7,  /* collective source/dest ranges partially overlap              */
    SHMEMG_ERR_NODEVICE = -8  /* no sm_100 device / wrong architecture / peer GPU unreachable  */
};

/* ---- teams and contexts: constants only in this build ------------------ */
enum {
    SHMEM_TEAM_WORLD = 0,
    SHMEM_DEVICE_TEAM_WORLD = 1,    /* same membership as SHMEM_TEAM_WORLD            */
    SHMEM_DEVICE_TEAM_SHARED = 2    /* all PEs share one GPU, so shared == world here (L357)       */
};
#define SHMEM_DEVICE_CTX_DEFAULT 0   /* the one default device context = one ordering domain per PE */

/* ---- capability bits (shape left open by the paper) ------ */
#define SHMEMG_CAP_GPU_HEAP_PRESENT           (1ull << 0)   /* a GPU symmetric heap exists (L299)        */
#define SHMEMG_CAP_DEFAULT_HEAP_IS_GPU        (1ull << 1)   /* GPU-first: default heap type (L451)        */
#define SHMEMG_CAP_HOST_INITIATED_GPU_BUFFERS (1ull << 2)   /* Tier-0 baseline (L465)                    */
#define SHMEMG_CAP_STREAM_TRIGGERED           (1ull << 3)   /* _on_stream variants (L396, L412)          */
#define SHMEMG_CAP_DEVICE_INITIATED           (1ull << 4)   /* __device__ entry points (L412, L465)      */
#define SHMEMG_CAP_DEVICE_COLLECTIVES         (1ull << 5)   /* shmemg_dev_{sum_reduce,fcollect,alltoall,broadcast}_block (L226, L363) */
#define SHMEMG_CAP_EXPLICIT_DEVICE_CTX        (1ull << 6)   /* shmemg_ctx_create + shmemg_dev_*_nbi / shmemg_dev_ctx_* (L327, L331) */
#define SHMEMG_CAP_PTR_DEVICE_ACCESSIBLE      (1ull << 7)   /* shmemg_ptr is a device pointer (L353)     */
#define SHMEMG_CAP_PTR_HOST_ACCESSIBLE        (1ull << 8)   /* 0: not dereferenceable on the host (L456) */
#define SHMEMG_CAP_PROGRESS_GPU_ONLY          (1ull << 9)   /* no host proxy needed (L394, L431)         */
#define SHMEMG_CAP_PATH_DIRECT                (1ull << 10)  /* direct load/store path (L431)             */
#define SHMEMG_CAP_ATOMICS_64                 (1ull << 11)  /* add / fetch-add / compare-swap on 64 bit  */
#define SHMEMG_CAP_STREAM_COLLECTIVES         (1ull << 12)  /* barrier/alltoall/fcollect/reduce on stream */
#define SHMEMG_CAP_DEVICE_BARRIER             (1ull << 13)  /* shmemg_dev_barrier_all_block (L363)       */
#define SHMEMG_CAP_CPU_HEAP_PRESENT           (1ull << 14)  /* the CPU space of the two-space model is attached (L313-L317) */
#define SHMEMG_CAP_PEER_SHARDS                (1ull << 15)  /* this world is one shard of a multi-GPU world (shmemg_shard_init, L194) */

/* ---- lifecycle ------------------------------------------------------------------------------------ */

/* Bytes the caller must provide for the slab: npes heap windows (stride = heap_bytes_per_pe rounded up
 * to 512 B) plus the library's control region and plan arena (64 KiB + 4 MiB).  heap_bytes_per_pe == 0 means "take it from the
 * environment variable SHMEMG_SYMMETRIC_SIZE" (bytes, optional K/M/G suffix).
 * Returns 0 on invalid arguments. */
SHMEMG_API size_t shmemg_slab_bytes_required(int npes, size_t heap_bytes_per_pe);

/* Create a world of `npes` logical PEs over `device_slab` (DEVICE, 512-byte aligned, owned by the
 * caller, >= shmemg_slab_bytes_required bytes).  GPU-first: the GPU symmetric heap exists right after
 * init.  Zeroes the control region on the legacy default stream and synchronises.
 * *out receives the handle (HOST). */
SHMEMG_API int shmemg_init(int npes, size_t heap_bytes_per_pe, void *device_slab, size_t slab_bytes,
                           shmemg_world_t **out);
SHMEMG_API int shmemg_finalize(shmemg_world_t *w);
SHMEMG_API int shmemg_n_pes(const shmemg_world_t *w);
SHMEMG_API size_t shmemg_heap_bytes(const shmemg_world_t *w);    /* usable bytes per PE           */
SHMEMG_API size_t shmemg_heap_stride(const shmemg_world_t *w);   /* distance between PE windows   */
/* Text of the last SHMEMG_ERR_CUDA on this world; also the reason when shmemg_atomic_fetch_add_batch_static_on_stream refuses a call. */
SHMEMG_API const char *shmemg_last_cuda_error(const shmemg_world_t *w);

/* Capability discovery ("shmem_query_capabilities", section 6.5).  `team` is one of the
 * SHMEM_*TEAM* constants; *caps (HOST) receives the SHMEMG_CAP_* mask active for that team. */
SHMEMG_API int shmem_query_capabilities(const shmemg_world_t *w, int team, uint64_t *caps);

/* ---- symmetric allocation in the GPU space ("shmemg_malloc") ---------------------------
 * One call allocates on ALL PEs (one process owns all PEs, so the call is collective by construction)
 * and yields ONE offset valid on every PE; allocation order and size are symmetric (L303).  Alignment
 * >= 256 B.  Contents are unspecified after malloc/align, zero after calloc (enqueued on `stream`). */
SHMEMG_API int shmemg_malloc(shmemg_world_t *w, size_t bytes, uint64_t *sym_off);
SHMEMG_API int shmemg_calloc(shmemg_world_t *w, size_t count, size_t size, uint64_t *sym_off, void *stream);
SHMEMG_API int shmemg_align(shmemg_world_t *w, size_t alignment, size_t bytes, uint64_t *sym_off);
SHMEMG_API int shmemg_free(shmemg_world_t *w, uint64_t sym_off);
/* shmem_ptr analog: DEVICE pointer to offset `sym_off` on PE `pe`, or NULL if the
 * arguments are invalid.  Valid in the device access domain only (SHMEMG_CAP_PTR_DEVICE_ACCESSIBLE). */
SHMEMG_API void *shmemg_ptr(const shmemg_world_t *w, uint64_t sym_off, int pe);

/* ---- the two-space model (Fig. 4 "Two-space model (baseline)": a GPU space and a "CPU
 * space: default symmetric heap (host-attached)"; L456 access domains) ---------------------------------------------------------
 * The GPU space is the heap of shmemg_init.  shmemg_cpu_heap_attach adds the CPU space: npes windows of heap_bytes_per_pe bytes
 * (stride rounded up to 512 B) in `host_slab`, PAGE-LOCKED host memory owned by the caller (cudaHostAlloc / torch pin_memory;
 * SHMEMG_ERR_ARG otherwise), at most once per world.  shmemg_cpu_malloc / shmemg_cpu_free allocate symmetric offsets in it (its
 * own allocator: an offset names ONE space), shmemg_cpu_ptr is dereferenceable on the HOST.  shmemg_put_space_on_stream /
 * shmemg_get_space_on_stream are put / get whose dest and source each name their space: GPU <-> GPU runs the copy kernels,
 * anything that touches the CPU space is a DMA transfer on `stream`.  shmem_query_capabilities reports
 * SHMEMG_CAP_CPU_HEAP_PRESENT once it is attached; AMOs, signals and collectives stay in the GPU space. */
enum { SHMEMG_SPACE_GPU = 0, SHMEMG_SPACE_CPU = 1 };
SHMEMG_API int shmemg_cpu_heap_attach(shmemg_world_t *w, void *host_slab, size_t heap_bytes_per_pe, size_t slab_bytes);
SHMEMG_API int shmemg_cpu_malloc(shmemg_world_t *w, size_t bytes, uint64_t *sym_off);
SHMEMG_API int shmemg_cpu_free(shmemg_world_t *w, uint64_t sym_off);
SHMEMG_API void *shmemg_cpu_ptr(const shmemg_world_t *w, uint64_t sym_off, int pe);      /* HOST pointer, or NULL */
SHMEMG_API int shmemg_put_space_on_stream(shmemg_world_t *w, int dest_space, uint64_t dest_off, int source_space, uint64_t source_off,
                                          size_t nbytes, int pe, int target_pe, void *stream);
SHMEMG_API int shmemg_get_space_on_stream(shmemg_world_t *w, int dest_space, uint64_t dest_off, int source_space, uint64_t source_off,
                                          size_t nbytes, int pe, int target_pe, void *stream);

/* Documented extension ("registered private ... source operands"): move bytes between a HOST
 * buffer and PE `pe`'s window with cudaMemcpyAsync on `stream`.  Used by the end-to-end benchmark. */
SHMEMG_API int shmemg_heap_write_on_stream(shmemg_world_t *w, int pe, uint64_t dst_off, const void *src_host,
                                           size_t nbytes, void *stream);
SHMEMG_API int shmemg_heap_read_on_stream(shmemg_world_t *w, int pe, void *dst_host, uint64_t src_off,
                                          size_t nbytes, void *stream);

/* ---- op batches: host-initiated enqueue on a stream ------------------------ */

enum {
    SHMEMG_OP_PUT = 1,                  /* heap[target][rem_off..] = heap[initiator][loc_off..]   (L116) */
    SHMEMG_OP_GET = 2,                  /* heap[initiator][loc_off..] = heap[target][rem_off..]   (L116) */
    SHMEMG_OP_PUT_SIGNAL = 3,           /* PUT, then signal word sig_off on target SET/ADD `value` (L218, L461) */
    SHMEMG_OP_ATOMIC_ADD = 4,           /* u64 heap[target][rem_off] += value                      (L116) */
    SHMEMG_OP_ATOMIC_FETCH_ADD = 5,     /* as ADD; old value -> u64 heap[initiator][loc_off]       (L116) */
    SHMEMG_OP_ATOMIC_COMPARE_SWAP = 6,  /* if (*p == cond) *p = value; old -> heap[initiator][loc_off] (L361) */
    SHMEMG_OP_SIGNAL_WAIT_UNTIL = 7,    /* initiator blocks until cmp(u64 heap[initiator][loc_off], value) (L116, L392) */
    SHMEMG_OP_FENCE = 8,                /* orders initiator's later ops after its earlier ones      (L377) */
    SHMEMG_OP_QUIET = 9,                /* initiator's earlier ops complete and are visible         (L377-L390) */
    SHMEMG_OP_BARRIER_ALL = 10          /* all PEs: every earlier op of every PE complete           (L116, L369) */
};
#define SHMEMG_CTX_MAX 8
enum { SHMEMG_SIGNAL_SET = 0, SHMEMG_SIGNAL_ADD = 1 };
enum { SHMEMG_CMP_EQ = 0, SHMEMG_CMP_NE = 1, SHMEMG_CMP_GT = 2, SHMEMG_CMP_GE = 3, SHMEMG_CMP_LT = 4, SHMEMG_CMP_LE = 5 };

/* One op descriptor, 64 bytes, in HOST memory (shmemg_batch_create, shmemg_device_exec_ops_on_stream) or DEVICE memory
 * (shmemg_enqueue_batch).  "Remote" = the target PE's window, "local" = the initiator's window.  Unused fields are ignored. */
typedef struct shmemg_op {
    uint8_t opcode;        /* SHMEMG_OP_*                                                     */
    uint8_t sig_op;        /* SHMEMG_SIGNAL_* (PUT_SIGNAL)                                    */
    uint8_t cmp;           /* SHMEMG_CMP_*    (SIGNAL_WAIT_UNTIL), unsigned 64-bit comparison */
    uint8_t ctx;           /* context of the op, 0 .. SHMEMG_CTX_MAX-1 (0 = the default context): FENCE / QUIET /
                            * SIGNAL_WAIT_UNTIL order only ops of the same (PE, context) pair */
    int32_t initiator_pe;
    int32_t target_pe;
    uint32_t reserved1;
    uint64_t rem_off;      /* put dest / get source / AMO word, in the TARGET's window       */
    uint64_t loc_off;      /* put source / get dest / fetch slot / wait word, in the INITIATOR's window */
    uint64_t nbytes;       /* put / get / put_signal payload size; any size and alignment >= 0 */
    uint64_t value;        /* AMO operand, signal value, or wait comparand                    */
    uint64_t cond;         /* compare-swap condition                                          */
    uint64_t sig_off;      /* signal word in the TARGET's window (8-byte aligned)             */
} shmemg_op_t;

/*
 * Batch semantics:
 *   - ops[0..nops) is an ordered program; REQUIREMENT: index order is a valid sequential schedule (a
 *     SIGNAL_WAIT_UNTIL is satisfied by ops that precede it in the array).
 *   - ops have non-blocking semantics: the executor may run ops of one PE in any order and
 *     concurrently unless a FENCE / QUIET / SIGNAL_WAIT_UNTIL of that PE or a BARRIER_ALL lies between
 *     them.  FENCE and QUIET are both implemented as "all earlier ops of this PE, to all targets, gets
 *     and atomics included, are complete and visible before any later op of this PE starts" -- the
 *     strong reading of L377, always conformant.  A wait also orders the PE's later ops after it.
 *     "Of this PE" means: of the same (PE, ctx) pair -- contexts are independent ordering domains (L124-L130); a QUIET on
 *     context 1 does not wait for the PE's traffic on context 0.  BARRIER_ALL covers every context of every PE.
 *     This holds for SIGNAL_WAIT_UNTIL too, and there a batch is WEAKER than the device-initiated paths: a wait with ctx = c
 *     holds back only the later ops of (PE, c), whereas in shmemg_device_exec_ops(_ctx)_on_stream and for shmemg_dev_* calls
 *     the wait blocks the PE's whole agent, the way OpenSHMEM's shmem_wait_until blocks the calling PE.  An op list that waits
 *     on context c and then forwards the received data on another context c' is therefore ordered when device-initiated but
 *     not in a batch; portable lists repeat the wait (same word, same comparison) on c', or issue the dependent op on c.
 *   - PUT_SIGNAL: the signal update is atomic w.r.t. other signal updates and waits, and becomes visible
 *     only after the whole payload (release/acquire at GPU scope).
 *   - atomicity does not imply ordering.
 *   - batch end = kernel end = quiet for every PE + barrier (stronger than required; L377).
 */

/* DEVICE bytes needed for the plan of this op list (0 on invalid arguments). */
SHMEMG_API size_t shmemg_batch_plan_bytes(const shmemg_world_t *w, const shmemg_op_t *ops_host, size_t nops);

/* Validate `ops_host` (HOST, nops entries), resolve PE->address translation, cut the ops into tiles and
 * upload the plan into `plan_dev` (DEVICE, 256-byte aligned, >= shmemg_batch_plan_bytes, caller-owned,
 * must outlive the batch) on `stream`, then synchronise that stream.  On a bad descriptor returns the
 * error code and stores its index in *bad_index (HOST, may be NULL).  A batch may be enqueued any
 * number of times, but never concurrently with itself. */
SHMEMG_API int shmemg_batch_create(shmemg_world_t *w, const shmemg_op_t *ops_host, size_t nops, void *plan_dev,
                                   size_t plan_bytes, void *stream, shmemg_batch_t **out, size_t *bad_index);
SHMEMG_API int shmemg_batch_destroy(shmemg_batch_t *b);
/* Number of kernel launches one enqueue of this batch performs (for launch accounting). */
SHMEMG_API int shmemg_batch_launches(const shmemg_batch_t *b);

/* Launch the batch executor on `stream` (one persistent-grid kernel; tiles are claimed in batch order). */
SHMEMG_API int shmemg_batch_enqueue_on_stream(shmemg_world_t *w, shmemg_batch_t *b, void *stream);
/* Every executor launch (and the device planner of the one-call form) is by default a PROGRAMMATIC DEPENDENT of the kernel
 * before it on the stream, and every executor releases its own dependents when it starts: the next launch sets its CTAs up on
 * SMs as they become free and blocks until this one has completed (about 1 us per back-to-back launch).  Results never depend
 * on it.  Forward progress can: while an executor still polls SIGNAL_WAIT_UNTIL ops that only a kernel on ANOTHER stream (a
 * device-initiated sender) can satisfy, the parked CTAs of the next launch hold SMs that sender may need to become resident.
 * A caller that relies on such cross-stream senders turns the feature off for the world (enable = 0: plain stream-ordered
 * launches).  The environment variable SHMEMG_NO_PDL, read once in shmemg_init, sets the initial state to off. */
SHMEMG_API int shmemg_set_dependent_launch(shmemg_world_t *w, int enable);

/*
 * ONE-CALL FORM: host-initiated enqueue of a DEVICE-RESIDENT descriptor array ("on
 * stream", L335 "An implementation may use internal GPU kernels to accelerate a host-issued or stream-triggered operation",
 * L396).  `ops_dev` (DEVICE, 16-byte aligned, nops entries of shmemg_op_t, caller-owned, valid until the stream has passed
 * the call) is planned ON THE DEVICE by one internal kernel (validation, PE -> address translation, tile cutting, dependency
 * thresholds: the same plan shmemg_batch_create builds on the host) and executed by the batch executor launched behind it
 * as a programmatic dependent.  No host pass over the descriptors, no synchronisation; the descriptors may have been written
 * by earlier work on the stream (a kernel that generates the op list).  Batch semantics as above.
 *   - shmemg_enqueue_batch uses the world's plan arena (4 MiB carved from the slab behind the control region; it holds a
 *     batch of about 16 000 ops / 40 000 tile records).  Two calls that use the arena must be stream-ordered.
 *   - shmemg_enqueue_batch_ws takes the workspace from the caller: `work_dev` (DEVICE, 256-byte aligned, work_bytes >=
 *     shmemg_batch_work_bytes(w, nops, payload) where payload is an upper bound of the sum of the nbytes fields; valid until
 *     the stream has passed the call; may be reused by a later call on the same stream).
 *   Host-checkable misuse (NULL, alignment, a workspace too small for nops records) returns an error and enqueues nothing.
 *   What only the device can see is reported in the plan header and nothing of the batch is executed: the first invalid
 *   descriptor (same checks and codes as shmemg_batch_create), or SHMEMG_ERR_NOMEM when the tile records do not fit the
 *   workspace.  shmemg_batch_status reads that status back (work_dev NULL = the arena; synchronises `stream`; *bad_index =
 *   index of the bad descriptor, or the number of tile records needed).  More than 512 PEs: SHMEMG_ERR_ARG (plan on the host).
 */
SHMEMG_API size_t shmemg_batch_work_bytes(const shmemg_world_t *w, size_t nops, uint64_t payload_bytes);
SHMEMG_API int shmemg_enqueue_batch(shmemg_world_t *w, const shmemg_op_t *ops_dev, size_t nops, void *stream);
SHMEMG_API int shmemg_enqueue_batch_ws(shmemg_world_t *w, const shmemg_op_t *ops_dev, size_t nops, void *work_dev,
                                       size_t work_bytes, void *stream);
SHMEMG_API int shmemg_batch_status(shmemg_world_t *w, const void *work_dev, void *stream, int *status, size_t *bad_index);

/* ---- single operations on a stream (put/get, signal put/wait, barrier on stream) ------ */
SHMEMG_API int shmemg_put_on_stream(shmemg_world_t *w, uint64_t dest_off, uint64_t source_off, size_t nbytes,
                                    int pe /*initiator*/, int target_pe, void *stream);
SHMEMG_API int shmemg_get_on_stream(shmemg_world_t *w, uint64_t dest_off, uint64_t source_off, size_t nbytes,
                                    int pe /*initiator*/, int target_pe, void *stream);
SHMEMG_API int shmemg_put_signal_on_stream(shmemg_world_t *w, uint64_t dest_off, uint64_t source_off, size_t nbytes,
                                           uint64_t sig_off, uint64_t signal, int sig_op, int pe, int target_pe,
                                           void *stream);
/* Blocks the STREAM (not the host) until cmp(u64 heap[pe][sig_off], value).  Only ops enqueued EARLIER on
 * the same stream, or device-initiated ops, can satisfy it (prohibited pattern otherwise). */
SHMEMG_API int shmemg_signal_wait_until_on_stream(shmemg_world_t *w, uint64_t sig_off, int cmp, uint64_t value,
                                                  int pe, void *stream);
/* Stream order already completes every earlier `_on_stream` op before a later one starts, so these
 * validate their arguments and enqueue nothing (ordering within a stream). */
SHMEMG_API int shmemg_fence_on_stream(shmemg_world_t *w, int pe, void *stream);
SHMEMG_API int shmemg_quiet_on_stream(shmemg_world_t *w, int pe, void *stream);
/* Host-blocking quiet: stream-ordered quiet + cudaStreamSynchronize. */
SHMEMG_API int shmemg_quiet(shmemg_world_t *w, int pe, void *stream);

/* ---- homogeneous AMO batches, structure-of-arrays (PAPER L116, L224 case study 2) ---------------------
 * Op i targets 64-bit word  heap[tgt_pe[i]][sym_off + 8*elem_idx[i]].  tgt_pe, elem_idx, val, cond and
 * fetched_out are DEVICE arrays of n entries; elem_idx has `idx_bytes` (4 or 8) bytes per entry; `val` /
 * `cond` may be NULL, in which case `val_scalar` / `cond_scalar` is used for every op (immediates, L355).
 * There is NO ordering between the ops of one call (reading 7); fetched values are valid when the stream
 * has passed the call.  flags: SHMEMG_AMO_* below.  64-bit integer types only (wraparound add). */
#define SHMEMG_AMO_WARP_AGGREGATE 1u   /* combine same-address ops of a warp into one L2 atomic */
/* compare-swap with a scalar cond only: read the word first and issue the L2 atomic only while the word may still equal
 * cond.  Legal because the ops of one call are unordered and each swaps only cond -> val: once a word differs from cond no
 * op of the call can change it, so the loaded value is the failed swap's fetched value (the load may be served by the SM's
 * L1, which is empty when the call starts: a value found there was the word's value at some instant of this call; a stale
 * cond is decided by the L2 atomic that follows).  The op's val is read only when the atomic is issued.
 * Requires that nothing outside this call updates the target words while it runs (already undefined). */
#define SHMEMG_AMO_TEST_BEFORE_SWAP 2u
/* add / fetch-add with a scalar value (val == NULL), meant for skewed streams (same-line serialisation at the L2 atomic
 * unit is the limiter there): a sampling kernel finds the hot words of the stream (up to 512); in the main kernel every CTA
 * combines its ops on a hot word in shared memory and issues ONE L2 atomic per hot word (op k of the CTA's group fetches
 * old + k*val_scalar: the group executes back to back, legal for the same reason as warp aggregation).  The sample only
 * affects speed, never the result.  Uses scratch in the world's control region and the caller-owned scratch buffer registered with
 * shmemg_set_scratch (>= shmemg_amo_scratch_bytes(w, n)); two calls with this flag must be stream-ordered.  Ignored (the plain
 * kernel runs) when no large enough scratch buffer is registered, val != NULL, n < 2^20 or n >= 2^33, or the slab has 2^32 or
 * more 64-bit words. */
#define SHMEMG_AMO_HOT_AGGREGATE 4u
/* quiet for every PE + barrier_all folded into the same launch (config C1 ends with "quiet + barrier"): the end of the kernel
 * completes every AMO of the call and orders it before later work on the stream; the CTA that finishes last bumps the world's
 * barrier epoch, exactly what a following shmemg_barrier_all_on_stream would have done with a second launch. */
#define SHMEMG_AMO_THEN_BARRIER 8u
/* Caller-owned DEVICE scratch (256-byte aligned) for the calls that need some (SHMEMG_AMO_HOT_AGGREGATE); the library itself
 * never allocates device memory.  Valid until replaced (scratch_dev NULL: none) or shmemg_finalize; calls that use it must be
 * stream-ordered.  shmemg_amo_scratch_bytes: what a SHMEMG_AMO_HOT_AGGREGATE call of n ops needs. */
SHMEMG_API size_t shmemg_amo_scratch_bytes(const shmemg_world_t *w, size_t n);
SHMEMG_API int shmemg_set_scratch(shmemg_world_t *w, void *scratch_dev, size_t bytes);
/* Which kernels the world's LAST shmemg_atomic_add_batch_on_stream / shmemg_atomic_fetch_add_batch_on_stream call enqueued:
 * 1 = the hot-set kernels (SHMEMG_AMO_HOT_AGGREGATE honoured), 0 = the plain kernel (flag absent, or ignored for one of the
 * reasons listed above, or the sampling CTAs could not be made co-resident).  The result is the same either way; a benchmark
 * asks so that a number is never attributed to the wrong kernel. */
SHMEMG_API int shmemg_amo_last_path(const shmemg_world_t *w);
SHMEMG_API int shmemg_atomic_add_batch_on_stream(shmemg_world_t *w, uint64_t sym_off, const int32_t *tgt_pe,
                                                 const void *elem_idx, int idx_bytes, const uint64_t *val,
                                                 uint64_t val_scalar, size_t n, uint32_t flags, void *stream);
SHMEMG_API int shmemg_atomic_fetch_add_batch_on_stream(shmemg_world_t *w, uint64_t sym_off, const int32_t *tgt_pe,
                                                       const void *elem_idx, int idx_bytes, const uint64_t *val,
                                                       uint64_t val_scalar, uint64_t *fetched_out, size_t n,
                                                       uint32_t flags, void *stream);
SHMEMG_API int shmemg_atomic_compare_swap_batch_on_stream(shmemg_world_t *w, uint64_t sym_off, const int32_t *tgt_pe,
                                                          const void *elem_idx, int idx_bytes, const uint64_t *cond,
                                                          uint64_t cond_scalar, const uint64_t *val,
                                                          uint64_t val_scalar, uint64_t *fetched_out, size_t n,
                                                          uint32_t flags, void *stream);

/* ---- fetch-add for callers that cannot allocate device memory ------------------------------------------------------------
 * The fast fetch-add on skewed streams (SHMEMG_AMO_HOT_AGGREGATE above) needs device scratch, and everywhere else in this
 * library the caller provides it (shmemg_set_scratch).  Some callers have no way to get any: a plug-in or callback that a host
 * runtime hands a stream, the slab and its input / output pointers but not its allocator; a process that gave all of the
 * GPU's memory to one pool at start-up, so that a later cudaMalloc fails; a caller inside a latency-critical stream pipeline,
 * where cudaMalloc / cudaFree would synchronise the whole device.  This entry point is for them.  It computes exactly what
 *     shmemg_atomic_fetch_add_batch_on_stream(w, sym_off, tgt_pe, elem_idx, idx_bytes, NULL, val_scalar, fetched_out, n,
 *                                             flags | SHMEMG_AMO_HOT_AGGREGATE, stream)
 * computes (same kernels, same result contract: per word the fetched values are the prefix sums of some order of the
 * word's ops, the final words are exact), but the scratch of the hot-set kernels is an array that is part of the library
 * image: SHMEMG_STATIC_SCRATCH_BYTES of device memory on EVERY GPU on which this library is loaded, held until the process
 * exits, whether or not this call is ever made.  The call itself calls no cudaMalloc / cudaFree and no allocating library
 * routine; inputs (tgt_pe, elem_idx) and the output (fetched_out) are still the caller's DEVICE arrays of n entries.
 *   Limit: n <= SHMEMG_STATIC_MAX_OPS.  A larger n is refused with SHMEMG_ERR_NOMEM before anything is launched, and
 *     shmemg_last_cuda_error(w) then holds a sentence naming n and the limit (split the batch, or use shmemg_set_scratch).
 *   flags: SHMEMG_AMO_THEN_BARRIER and SHMEMG_AMO_HOT_AGGREGATE (implied) only; any other bit is SHMEMG_ERR_ARG.
 *   The world's device must be the CURRENT device of the calling thread (SHMEMG_ERR_ARG otherwise).
 *   First call per device: it looks the array's device address up (cudaGetSymbolAddress, once per device, remembered for
 *     the life of the process).  Make that first call during set-up, before any stream capture is begun.
 *   Sharing: there is ONE array per GPU, shared by every call on every world of that GPU, and it keeps whatever the
 *     previous call left in it.  Nothing in it has to start at zero (each call writes every scratch word before it reads it,
 *     so no clearing pass runs), but two calls that can overlap in time on the GPU -- different streams, different worlds,
 *     different host threads -- corrupt each other's hot-op lists: keep all calls on a device stream-ordered.
 *   When the hot-set kernels do not apply (n < 2^20, a slab of 2^32 or more 64-bit words, or the 16 sampling CTAs cannot be
 *     made co-resident) the plain fetch-add kernel runs instead; it needs no scratch at all.  *path_out (HOST, may be NULL)
 *     says which one ran: 1 = hot-set kernels on the built-in scratch, 0 = plain kernel. */
#define SHMEMG_STATIC_SCRATCH_BYTES (8u << 20)
#define SHMEMG_STATIC_MAX_OPS ((size_t)1 << 22)
SHMEMG_API int shmemg_atomic_fetch_add_batch_static_on_stream(shmemg_world_t *w, uint64_t sym_off, const int32_t *tgt_pe,
                                                              const void *elem_idx, int idx_bytes, uint64_t val_scalar,
                                                              uint64_t *fetched_out, size_t n, uint32_t flags,
                                                              void *stream, int *path_out);

/* Generic AMO batch on `width`-byte words (4 or 8), structure-of-arrays like the calls above (the AMO set of OpenSHMEM 1.6,
 * inherited unchanged): word = heap[tgt_pe[i]][sym_off + width*elem_idx[i]]; old = word; word = f(old, val[i]);
 * fetched_out[i] = old when fetched_out != NULL (zero-extended to 64 bits).  ADD / AND / OR / XOR; SWAP (word = val;
 * with fetched_out == NULL this is atomic_set); FETCH (atomic read, fetched_out required, val ignored).  inc / fetch_inc
 * are ADD with val_scalar = 1.  `val` (DEVICE, 64-bit entries, low `width` bytes used) may be NULL -> val_scalar.
 * Non-fetching ops use red.global / st, fetching ops atom.global / ld.  No ordering between the ops of one call. */
enum { SHMEMG_AMO_ADD = 0, SHMEMG_AMO_AND = 1, SHMEMG_AMO_OR = 2, SHMEMG_AMO_XOR = 3, SHMEMG_AMO_SWAP = 4,
       SHMEMG_AMO_FETCH = 5 };
SHMEMG_API int shmemg_atomic_op_batch_on_stream(shmemg_world_t *w, int amo, int width, uint64_t sym_off,
                                                const int32_t *tgt_pe, const void *elem_idx, int idx_bytes,
                                                const uint64_t *val, uint64_t val_scalar, uint64_t *fetched_out,
                                                size_t n, void *stream);

/* compare-swap of the same AMO set on `width`-byte words (4 or 8): old = word; if (old == cond[i]) word = val[i];
 * fetched_out[i] = old (required; zero-extended).  cond / val (DEVICE, 64-bit entries, low `width` bytes used) may be NULL ->
 * cond_scalar / val_scalar.  atom.global.cas.b32 / .b64; no ordering between the ops of one call.  (The 64-bit claim-style
 * batches of config 4 have their own faster call above, shmemg_atomic_compare_swap_batch_on_stream.) */
SHMEMG_API int shmemg_atomic_cswap_op_batch_on_stream(shmemg_world_t *w, int width, uint64_t sym_off, const int32_t *tgt_pe,
                                                      const void *elem_idx, int idx_bytes, const uint64_t *cond,
                                                      uint64_t cond_scalar, const uint64_t *val, uint64_t val_scalar,
                                                      uint64_t *fetched_out, size_t n, void *stream);

/* Debug aid for every structure-of-arrays AMO call above.  Their tgt_pe[] / elem_idx[] are DEVICE arrays, so per-op bounds are
 * the caller's contract and a bad entry is undefined behaviour: a stray atomic.  This call checks them on the
 * device with the same addressing (word = heap[tgt_pe[i]][sym_off + width*elem_idx[i]], width 4 or 8; pass 8 for the 64-bit
 * add / fetch-add / compare-swap calls): *first_bad_dev (DEVICE, 8 bytes, caller-owned) receives the smallest i whose PE is
 * outside [0, npes) or whose word is not wholly inside the PE's heap window, or UINT64_MAX when every op is in bounds.  Valid
 * when `stream` has passed the call (one 8-byte memset + one kernel; reads 4 + idx_bytes bytes per op). */
SHMEMG_API int shmemg_amo_check_batch_on_stream(shmemg_world_t *w, int width, uint64_t sym_off, const int32_t *tgt_pe,
                                                const void *elem_idx, int idx_bytes, size_t n, uint64_t *first_bad_dev,
                                                void *stream);

/* ---- block-strided put / get (OpenSHMEM 1.6 ibput / ibget; iput / iget are the case block = one element) ---------------
 * for b in [0, nblocks): dest[b*dst_stride .. +block_bytes) = source[b*src_stride .. +block_bytes); strides in BYTES, any
 * size and alignment.  put: source in `pe`'s window, dest in `target_pe`'s; get: source in `target_pe`'s, dest in `pe`'s.
 * Destination blocks must not overlap each other (dst_stride < block_bytes with nblocks > 1: SHMEMG_ERR_OVERLAP) or the source
 * (undefined otherwise).  Stream-ordered like put / get. */
SHMEMG_API int shmemg_ibput_on_stream(shmemg_world_t *w, uint64_t dest_off, uint64_t source_off, uint64_t dst_stride,
                                      uint64_t src_stride, size_t block_bytes, size_t nblocks, int pe, int target_pe,
                                      void *stream);
SHMEMG_API int shmemg_ibget_on_stream(shmemg_world_t *w, uint64_t dest_off, uint64_t source_off, uint64_t dst_stride,
                                      uint64_t src_stride, size_t block_bytes, size_t nblocks, int pe, int target_pe,
                                      void *stream);

/* Vector forms on `nelems` consecutive u64 words of `pe`'s window starting at sig_off (OpenSHMEM 1.6 test_all / any / some and
 * wait_until_all / any / some).  The satisfied positions (ascending) go to indices_dev[0 .. count) and their
 * number to *count_dev (DEVICE uint64 arrays of nelems and 1 entries; either may be NULL), valid when the stream has passed the
 * call.  test_vec never blocks: all = (count == nelems), any = (count > 0, indices_dev[0] the lowest), some = the list.
 * wait_until_all blocks the stream until every word satisfies; wait_until_some (= wait_until_any: take indices_dev[0]) until
 * at least one does and reports those that do at that moment.  A satisfied word is an acquire.  Same prohibited stream
 * patterns as signal_wait_until_on_stream. */
SHMEMG_API int shmemg_signal_test_vec_on_stream(shmemg_world_t *w, uint64_t sig_off, size_t nelems, int cmp, uint64_t value,
                                                int pe, uint64_t *indices_dev, uint64_t *count_dev, void *stream);
SHMEMG_API int shmemg_signal_wait_until_all_on_stream(shmemg_world_t *w, uint64_t sig_off, size_t nelems, int cmp,
                                                      uint64_t value, int pe, void *stream);
SHMEMG_API int shmemg_signal_wait_until_some_on_stream(shmemg_world_t *w, uint64_t sig_off, size_t nelems, int cmp,
                                                       uint64_t value, int pe, uint64_t *indices_dev, uint64_t *count_dev,
                                                       void *stream);

/* ---- teams ("PE collectives remain collective over a team of PEs", L357, L412) --------
 * shmemg_team_split_strided: the PEs { start + k*stride : k < size } of `parent_team` (ranks of the parent; the three
 * predefined teams are the world) form a new team; *new_team receives its handle (>= SHMEMG_TEAM_USER0).  Team rank k is the
 * k-th member.  Teams live until shmemg_finalize.  The team collectives below are the world collectives with "all PEs"
 * replaced by "all members in team-rank order"; windows of non-members are untouched; `root_rank` is a TEAM rank.  They run
 * the same kernels on a strided view of the slab (member k's window = base + (start + k*stride) * heap_stride).
 * shmem_query_capabilities accepts user team handles and answers as for SHMEM_TEAM_WORLD. */
#define SHMEMG_TEAM_USER0 16
SHMEMG_API int shmemg_team_split_strided(shmemg_world_t *w, int parent_team, int start, int stride, int size, int *new_team);
SHMEMG_API int shmemg_team_n_pes(const shmemg_world_t *w, int team);
SHMEMG_API int shmemg_team_translate_pe(const shmemg_world_t *w, int team, int rank);     /* world PE of a team rank, or < 0 */
SHMEMG_API int shmemg_team_reduce_on_stream(shmemg_world_t *w, int team, int op, int dtype, uint64_t dest_off,
                                            uint64_t source_off, size_t nreduce, void *stream);
SHMEMG_API int shmemg_team_fcollect_on_stream(shmemg_world_t *w, int team, uint64_t dest_off, uint64_t source_off,
                                              size_t nbytes, void *stream);
SHMEMG_API int shmemg_team_alltoall_on_stream(shmemg_world_t *w, int team, uint64_t dest_off, uint64_t source_off,
                                              size_t nbytes, void *stream);
SHMEMG_API int shmemg_team_broadcast_on_stream(shmemg_world_t *w, int team, uint64_t dest_off, uint64_t source_off,
                                               size_t nbytes, int root_rank, void *stream);

/* signal test ("quiet, wait, and test"): *result_dev (DEVICE int32) = 1 if cmp(u64 heap[pe][sig_off], value)
 * holds when the stream reaches the call, else 0; never blocks.  A result of 1 is an acquire: work enqueued later on the
 * stream sees the payload the signal announced. */
SHMEMG_API int shmemg_signal_test_on_stream(shmemg_world_t *w, uint64_t sig_off, int cmp, uint64_t value, int pe,
                                            int32_t *result_dev, void *stream);

/* ---- collectives on SHMEM_TEAM_WORLD, one kernel each --------------------------
 * Each collective is one atomic unit in stream order (kernel boundaries order it against its neighbours). */
enum { SHMEMG_F32 = 0, SHMEMG_I64 = 1, SHMEMG_I32 = 2, SHMEMG_F64 = 3 };
/* every PE's dest[k] = sum over all PEs (ascending PE order) of source[k], k < nreduce.  F32 accumulates
 * in fp64 and rounds once; I64 wraps.  dest == source (exact aliasing) is allowed; partial overlap is not. */
SHMEMG_API int shmemg_sum_reduce_on_stream(shmemg_world_t *w, int dtype, uint64_t dest_off, uint64_t source_off,
                                           size_t nreduce, void *stream);
/* General reduction (the reduction set OpenSHMEM 1.6 defines, inherited unchanged):
 * every PE's dest[k] = op over all PEs (ascending PE order) of source[k].  SUM / PROD: fp32 accumulates in fp64 and rounds
 * once, fp64 accumulates in fp64, integers wrap.  MIN / MAX: signed for I32 / I64; floating-point inputs must be NaN-free.
 * AND / OR / XOR: I32 / I64 only (SHMEMG_ERR_ARG on F32 / F64).  Aliasing rules as for sum_reduce. */
enum { SHMEMG_RED_SUM = 0, SHMEMG_RED_PROD = 1, SHMEMG_RED_MIN = 2, SHMEMG_RED_MAX = 3, SHMEMG_RED_AND = 4,
       SHMEMG_RED_OR = 5, SHMEMG_RED_XOR = 6 };
SHMEMG_API int shmemg_reduce_on_stream(shmemg_world_t *w, int op, int dtype, uint64_t dest_off, uint64_t source_off,
                                       size_t nreduce, void *stream);
/* broadcast (named among the stream-ordered collectives; team-based form): every PE's dest[0 .. nbytes),
 * the root's included, = the root's source[0 .. nbytes).  Any size and alignment; source and dest ranges must not
 * overlap (SHMEMG_ERR_OVERLAP). */
SHMEMG_API int shmemg_broadcast_on_stream(shmemg_world_t *w, uint64_t dest_off, uint64_t source_off, size_t nbytes,
                                          int root_pe, void *stream);
/* every PE's dest[p*nbytes .. +nbytes) = PE p's source[0 .. nbytes)  (concatenation in PE order). */
SHMEMG_API int shmemg_fcollect_on_stream(shmemg_world_t *w, uint64_t dest_off, uint64_t source_off, size_t nbytes,
                                         void *stream);
/* PE j's dest[i*nbytes .. +nbytes) = PE i's source[j*nbytes .. +nbytes)  (block index = peer PE). */
SHMEMG_API int shmemg_alltoall_on_stream(shmemg_world_t *w, uint64_t dest_off, uint64_t source_off, size_t nbytes,
                                         void *stream);
/* Block-strided alltoall (the transposes of "FFT-driven spectral phases, many-to-many exchanges", PAPER L68;
 * generalises OpenSHMEM 1.6 alltoalls, inherited unchanged, L361): for all source PEs i, destination PEs j and blocks b < nblocks
 *     PE j's dest[i*dst_pe_stride + b*dst_block_stride .. +block_bytes) = PE i's source[j*src_pe_stride + b*src_block_stride .. +block_bytes)
 * (strides in BYTES).  A slab transpose of A[X][Y][Z] over N PEs is block = (Y/N)*Z*es, nblocks = X/N, src_block_stride = Y*Z*es,
 * src_pe_stride = block, dst_block_stride = block, dst_pe_stride = nblocks*block; alltoalls(dest, source, dst, sst, nelems) on
 * es-byte elements is block = es, nblocks = nelems, block strides dst*es / sst*es, pe strides nelems times those.  Any size and
 * alignment; the source and destination footprints must not overlap, nor two destination blocks (SHMEMG_ERR_OVERLAP where the
 * strides make it certain, undefined otherwise). */
SHMEMG_API int shmemg_alltoalls_on_stream(shmemg_world_t *w, uint64_t dest_off, uint64_t source_off, uint64_t dst_pe_stride,
                                          uint64_t src_pe_stride, uint64_t dst_block_stride, uint64_t src_block_stride,
                                          size_t block_bytes, size_t nblocks, void *stream);
/* Stream-level barrier: everything enqueued earlier on `stream` by any PE is complete and visible to
 * everything enqueued later; bumps the world's barrier epoch (one tiny kernel). */
SHMEMG_API int shmemg_barrier_all_on_stream(shmemg_world_t *w, void *stream);
/* `count` back-to-back barriers among npes co-resident PE agents (one CTA per PE, cooperative launch) in
 * ONE kernel: the in-kernel barrier whose per-iteration latency config C5 reports.  If `stamp_off` is not
 * UINT64_MAX, the agents also run the round-stamp check of SURVEY.md 8(c): in round r agent p writes r into
 * u64 heap[(p+1)%npes][stamp_off + 8*(r&1)], barrier, reads its own slot and counts a violation in
 * u64 heap[p][stamp_off + 16] if it is not r.  The object at stamp_off is 24 bytes, zero-initialised. */
SHMEMG_API int shmemg_barrier_all_repeat_on_stream(shmemg_world_t *w, uint32_t count, uint64_t stamp_off,
                                                   void *stream);
SHMEMG_API uint64_t shmemg_barrier_epoch(shmemg_world_t *w, void *stream);   /* synchronises `stream` */
/* Recovery.  The in-kernel barriers (shmemg_barrier_all_repeat_on_stream, shmemg_dev_barrier_all_block and the device
 * collectives built on it) and the sampling kernel of SHMEMG_AMO_HOT_AGGREGATE count arrivals in monotonic counters and find
 * their round from the count alone, which requires every kernel to finish its rounds.  After one that did not -- an aborted or
 * timed-out kernel, or a user kernel in which fewer than npes blocks reached a barrier -- every later barrier of the world
 * would release early, silently.  This call (one tiny kernel on `stream`; nothing of the world may be running concurrently)
 * rounds those counters up to the next round boundary and clears the last-arriver counters of put_signal / the AMO barrier
 * fold.  Harmless when nothing was wrong. */
SHMEMG_API int shmemg_realign_counters_on_stream(shmemg_world_t *w, void *stream);

/* ---- device-initiated path (Tier-1) ---------------------------------------------------
 * include/shmemg_device.cuh holds header-only `__device__` entry points (put/get/put_signal/wait/test/AMOs/fence/quiet
 * at thread, warp and block scope, and a block-scope barrier_all).  A kernel that uses them takes this POD BY VALUE. */
typedef struct shmemg_device_world {
    unsigned char *base;        /* DEVICE: window of PE 0                                                     */
    uint64_t stride;            /* distance between PE windows: address(pe, off) = base + pe*stride + off     */
    uint64_t heap_bytes;        /* usable bytes per PE                                                        */
    int32_t npes;
    int32_t reserved;
    unsigned long long *bar_arrivals;  /* DEVICE: device-barrier arrival counter (control region): monotonic, never reset */
    void *reserved2;
} shmemg_device_world_t;
/* Fill *out (HOST) for world w; valid until shmemg_finalize. */
SHMEMG_API int shmemg_device_world_get(const shmemg_world_t *w, shmemg_device_world_t *out);

/* ---- explicit device contexts ("explicit contexts as an advanced option", L331 "host-
 * created contexts that may be cached in GPU-accessible memory for later use by kernels") -------------------------------------
 * A context belongs to ONE PE and is an independent ordering / completion domain of that PE's device-initiated operations: it
 * owns a queue of pending NON-BLOCKING operations and its own completion counters (issued, completed).  The host creates it in
 * caller-owned DEVICE memory and receives a POD handle that kernels take BY VALUE (or read from device memory); see the `_nbi`
 * and `shmemg_dev_ctx_*` entry points of shmemg_device.cuh:
 *   - shmemg_dev_put_nbi / get_nbi / put_signal_nbi return before LOCAL completion: the transfer is recorded in
 *     the context and performed no later than the context's next quiet / fence, the PE's next barrier, or the next time the PE
 *     blocks (wait): the source must not change and a get's data must not be read until shmemg_dev_ctx_quiet has returned;
 *   - shmemg_dev_ctx_quiet(ctx) completes the operations of THAT context only; a quiet on another context of the same PE leaves
 *     them pending (their counters do not move);
 *   - the operations without a context argument keep using SHMEM_DEVICE_CTX_DEFAULT, which has no queue (they are blocking).
 * One thread (or one thread block, with uniform participation) uses a context at a time. */
typedef struct shmemg_nbi_rec {      /* 64 B: one pending non-blocking operation, addresses resolved */
    uint64_t dst, src, nbytes;
    uint64_t sig;                    /* put_signal: signal word (0 = none) */
    uint64_t sig_value;
    uint32_t sig_op, pad0;
    uint64_t pad1[2];
} shmemg_nbi_rec_t;
typedef struct shmemg_device_ctx {
    shmemg_nbi_rec_t *queue;         /* DEVICE: ring of `capacity` records                                      */
    unsigned long long *counters;    /* DEVICE: [0] = operations issued, [1] = operations completed (monotonic)  */
    uint32_t capacity;
    int32_t pe;                      /* the PE this context belongs to (the initiator of its operations)         */
} shmemg_device_ctx_t;
/* DEVICE bytes a context with a queue of `queue_entries` pending operations needs (0 on bad arguments). */
SHMEMG_API size_t shmemg_ctx_bytes(uint32_t queue_entries);
/* Create a context for PE `pe` in ctx_mem_dev (DEVICE, 256-byte aligned, >= shmemg_ctx_bytes, caller-owned, must outlive every
 * kernel that uses the handle); its counters are zeroed on `stream`.  *out (HOST) receives the handle. */
SHMEMG_API int shmemg_ctx_create(shmemg_world_t *w, int pe, uint32_t queue_entries, void *ctx_mem_dev, size_t ctx_mem_bytes,
                                 void *stream, shmemg_device_ctx_t *out);
/* Read the context's counters (synchronises `stream`): operations issued / completed so far. */
SHMEMG_API int shmemg_ctx_counters(shmemg_world_t *w, const shmemg_device_ctx_t *ctx, void *stream, uint64_t *issued,
                                   uint64_t *completed);
/* Like shmemg_device_exec_ops_on_stream, with explicit contexts: ctxs_dev is a DEVICE array of npes * nctx handles (entry
 * pe * nctx + c = context c of PE pe; every op's ctx field must be < nctx).  PUT / GET / PUT_SIGNAL are issued NON-BLOCKING on
 * their op's context, FENCE / QUIET act on that context only, AMOs are issued at once, a wait first progresses the PE's pending
 * operations (all its contexts), BARRIER_ALL and the end of the list complete everything (flags: SHMEMG_EXEC_*). */
#define SHMEMG_EXEC_LEAVE_PENDING 1u   /* no quiet at the end of the list: what is still queued stays pending in its context (contexts
                                        * live in device memory across kernels) until a later call completes it */
SHMEMG_API int shmemg_device_exec_ops_ctx_on_stream(shmemg_world_t *w, const shmemg_op_t *ops_host, size_t nops, void *ops_dev,
                                                    const shmemg_device_ctx_t *ctxs_dev, int nctx, uint32_t flags, void *stream,
                                                    size_t *bad_index);

/* ---- non-blocking forms on a stream ("For nonblocking operations ... completion only after an explicit quiet") ---
 * Host-issued, stream-ordered like shmemg_put_on_stream / shmemg_get_on_stream; the difference is the contract: a blocking
 * `_on_stream` put is locally complete for every LATER operation on the stream, a `_nbi` one only after the next
 * shmemg_quiet_on_stream / shmemg_quiet / shmemg_barrier_all_on_stream of that stream.  In this implementation stream order
 * already provides both, so the two forms launch the same kernels; programs that need the weaker contract only can say so. */
SHMEMG_API int shmemg_put_nbi_on_stream(shmemg_world_t *w, uint64_t dest_off, uint64_t source_off, size_t nbytes, int pe,
                                        int target_pe, void *stream);
SHMEMG_API int shmemg_get_nbi_on_stream(shmemg_world_t *w, uint64_t dest_off, uint64_t source_off, size_t nbytes, int pe,
                                        int target_pe, void *stream);
SHMEMG_API int shmemg_put_signal_nbi_on_stream(shmemg_world_t *w, uint64_t dest_off, uint64_t source_off, size_t nbytes,
                                               uint64_t sig_off, uint64_t signal, int sig_op, int pe, int target_pe, void *stream);

/* Run ONE device collective of include/shmemg_device.cuh device-initiated ("thread-collaborative
 * collective reductions ... device-callable collective operations", L363-L371 uniform participation): one cooperative kernel with
 * one thread block per PE; block p calls shmemg_dev_<kind>_block(..., pe = p) with the arguments given here.  kind:
 * SHMEMG_DEVCOLL_*; dtype (SUM_REDUCE only): SHMEMG_F32 / I64 / I32 / F64; n = nreduce (elements) or nbytes per block; root:
 * BROADCAST only.  Same results as the stream collectives (fp32 sums accumulate in fp64 in ascending PE order: bit-equal).
 * Returns SHMEMG_ERR_NOMEM if npes thread blocks cannot be co-resident. */
enum { SHMEMG_DEVCOLL_SUM_REDUCE = 0, SHMEMG_DEVCOLL_FCOLLECT = 1, SHMEMG_DEVCOLL_ALLTOALL = 2, SHMEMG_DEVCOLL_BROADCAST = 3 };
SHMEMG_API int shmemg_device_collective_on_stream(shmemg_world_t *w, int kind, int dtype, uint64_t dest_off, uint64_t source_off,
                                                  size_t n, int root, void *stream);

/* Run an op list DEVICE-INITIATED: one cooperative kernel with one thread block per PE ("PE agent"); agent p walks
 * ops[0..nops) in order and executes those it initiates through the entry points of shmemg_device.cuh with BLOCKING
 * semantics: put/get/put_signal at block scope, AMOs and fetch-slot stores by one thread, SIGNAL_WAIT_UNTIL
 * blocks the agent, FENCE/QUIET = shmemg_dev_quiet_block, BARRIER_ALL = shmemg_dev_barrier_all_block (executed by every
 * agent).  Same requirement as a batch: index order is a valid sequential schedule.  `ops_host` (HOST, nops entries) is
 * validated like shmemg_batch_create (error code returned, *bad_index set) and copied to `ops_dev` (DEVICE, >= 64*nops
 * bytes, caller-owned, must stay valid until the stream has passed the call) on `stream`.  Returns SHMEMG_ERR_NOMEM if
 * npes thread blocks cannot be co-resident on the device (progress would not be guaranteed). */
SHMEMG_API int shmemg_device_exec_ops_on_stream(shmemg_world_t *w, const shmemg_op_t *ops_host, size_t nops, void *ops_dev,
                                                void *stream, size_t *bad_index);

/* ---- PE -> GPU sharding over a load-store fabric ----------------------------------------
 * "Direct GPU-GPU fabrics such as NVLink ... load-store fabrics provide direct hardware-assisted communication among GPUs ...
 * They can offer high-performance remote atomic operations, but not necessarily in the same atomicity domain".
 * One process (one world) per GPU, G = nshards of them.  Placement (reading 42): GLOBAL PE g lives on shard
 * g mod G as that shard's LOCAL PE g div G; every shard holds `npes` local PEs (shmemg_init) with the same heap size, and the
 * symmetric allocator is called identically on every shard, so one offset names the same object everywhere.
 * The shards see each other's slabs through peer mappings: shmemg_shard_export gives a CUDA IPC handle of this world's slab
 * (64 bytes, HOST) plus the slab's byte offset inside the exported allocation; the caller carries both to the other processes
 * (any transport: the tests use torch.distributed/gloo) and gives them to shmemg_shard_attach_ipc there.  Shards that live in
 * ONE process pass the slab pointer itself to shmemg_shard_attach_ptr.  Both attach calls check that the peer slab is device
 * memory this world's GPU can reach: a slab on another GPU needs peer access (enabled here if it is not yet) over a link with
 * native atomics, since signals, the shard barrier and AMO batches update peer words with system-scope atomics; otherwise
 * SHMEMG_ERR_NODEVICE (reason in shmemg_last_cuda_error) and nothing is attached.  Status: this layer has been parity-tested
 * with all shards on ONE GPU only (in one process and as two processes over CUDA IPC); it has not yet run across NVLink.
 * The g-calls take GLOBAL PE numbers; the initiator must be a local PE of this shard.  Transfers are peer loads / stores issued
 * by this shard's kernels; AMOs and signal updates on a remote shard are SYSTEM-scope atomics (the atomicity domain of a
 * sharded world is the fabric, not one GPU's L2); ordering between shards comes from shmemg_gbarrier_all_on_stream or from
 * put-with-signal + wait, exactly as between PEs of one GPU.  shmemg_gbarrier_all_on_stream is one kernel per shard that
 * arrives on every shard's counter and waits for its own: the G kernels must be able to run at the same time (one GPU each);
 * it is a barrier of the STREAMS, so it also orders everything enqueued before it on each shard's stream.
 * shmemg_galltoall_on_stream: every local PE pushes its block for global PE j into j's window (peer stores), the caller puts a
 * gbarrier before it (sources ready) and after it (blocks delivered).
 * Errors: SHMEMG_ERR_ARG before shmemg_shard_init or for a shard that is not attached, SHMEMG_ERR_PE for a PE outside
 * [0, nshards * npes) or an initiator that is not local.  With nshards == 1 every g-call equals its unsharded counterpart. */
#define SHMEMG_MAX_SHARDS 16
SHMEMG_API int shmemg_shard_of(int gpe, int nshards);            /* g mod G, or SHMEMG_ERR_ARG */
SHMEMG_API int shmemg_shard_local_index(int gpe, int nshards);   /* g div G */
SHMEMG_API int shmemg_shard_global_pe(int shard, int local_pe, int nshards);
SHMEMG_API int shmemg_shard_init(shmemg_world_t *w, int nshards, int my_shard);
SHMEMG_API int shmemg_shard_export(shmemg_world_t *w, void *ipc_handle64_out, uint64_t *offset_out);
SHMEMG_API int shmemg_shard_attach_ipc(shmemg_world_t *w, int shard, const void *ipc_handle64, uint64_t offset);
SHMEMG_API int shmemg_shard_attach_ptr(shmemg_world_t *w, int shard, void *peer_slab_dev);
SHMEMG_API int shmemg_shard_global_npes(const shmemg_world_t *w);
SHMEMG_API int shmemg_gput_on_stream(shmemg_world_t *w, uint64_t dest_off, uint64_t source_off, size_t nbytes, int gpe,
                                     int target_gpe, void *stream);
SHMEMG_API int shmemg_gget_on_stream(shmemg_world_t *w, uint64_t dest_off, uint64_t source_off, size_t nbytes, int gpe,
                                     int target_gpe, void *stream);
SHMEMG_API int shmemg_gput_signal_on_stream(shmemg_world_t *w, uint64_t dest_off, uint64_t source_off, size_t nbytes,
                                            uint64_t sig_off, uint64_t signal, int sig_op, int gpe, int target_gpe, void *stream);
SHMEMG_API int shmemg_gsignal_wait_until_on_stream(shmemg_world_t *w, uint64_t sig_off, int cmp, uint64_t value, int gpe,
                                                   void *stream);
/* SoA AMO batches with GLOBAL target PEs (DEVICE arrays as in shmemg_atomic_*_batch_on_stream; the initiators are this shard's
 * PEs, which needs no argument: an AMO names only its target).  op: SHMEMG_OP_ATOMIC_ADD / _FETCH_ADD / _COMPARE_SWAP;
 * val == NULL: val_scalar for every op; cond likewise; fetched_out (DEVICE, n entries) for the two fetching ops. */
SHMEMG_API int shmemg_gatomic_batch_on_stream(shmemg_world_t *w, int op, uint64_t sym_off, const int32_t *target_gpe,
                                              const void *elem_idx, int idx_bytes, const uint64_t *cond, uint64_t cond_scalar,
                                              const uint64_t *val, uint64_t val_scalar, uint64_t *fetched_out, size_t n,
                                              void *stream);
SHMEMG_API int shmemg_galltoall_on_stream(shmemg_world_t *w, uint64_t dest_off, uint64_t source_off, size_t nbytes_per_pe,
                                          void *stream);
/* shmemg_gfcollect_on_stream: every local PE pushes its nbytes block into block g (its global number) of EVERY global PE's
 * dest.  shmemg_gsum_reduce_on_stream (dtype SHMEMG_F32 or SHMEMG_I64): an all-reduce over all global PEs computed as
 * reduce-scatter + all-gather over the fabric -- shard s reduces the s-th share of the nreduce elements over all the windows
 * (peer loads, ascending GLOBAL PE order, fp32 accumulated in fp64 and rounded once: bit-equal to the single-GPU routine and
 * to the oracle) and stores it into every PE's dest (peer stores).  source and dest must not overlap.  As for the alltoall,
 * the caller puts a gbarrier before (sources ready) and after (results delivered). */
SHMEMG_API int shmemg_gfcollect_on_stream(shmemg_world_t *w, uint64_t dest_off, uint64_t source_off, size_t nbytes, void *stream);
SHMEMG_API int shmemg_gsum_reduce_on_stream(shmemg_world_t *w, int dtype, uint64_t dest_off, uint64_t source_off, size_t nreduce,
                                            void *stream);
SHMEMG_API int shmemg_gbarrier_all_on_stream(shmemg_world_t *w, void *stream);

#ifdef __cplusplus
}
#endif
#endif /* SHMEMG_H */
