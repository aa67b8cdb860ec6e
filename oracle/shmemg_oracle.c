/*
 * oracle/shmemg_oracle.c -- CPU ORACLE.  TEST INFRASTRUCTURE, NOT PRODUCT.
 *
 * A plain, slow, single-threaded, sequential simulator of N logical PEs with
 * symmetric heaps, written from the paper (PAPER.md = /root/reference/PAPER.md at
 * build time; cited as "L<n>") and SURVEY.md section 8(c).  It shares no code,
 * header, table or helper with the CUDA path and neither imports the other.
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
 * reference legs may load this file.
 *
 * Nature of the result: none of these operations is an
 * approximation.  Each op has a plain definition (memcpy, integer add,
 * compare-and-swap, sum, concatenate, transpose); the oracle is that definition
 * written out, executed in BATCH INDEX ORDER, each op running to completion at its
 * turn.  That is one particular legal schedule under the paper's ordering rules
 * (L116, L126, L365-L369, L377-L390); outputs that may legitimately differ between
 * legal schedules (fetched values of fetch-add / compare-swap) are compared through
 * invariants in tests/, not through this schedule.
 *
 * Pins (tests/test_oracle_pins.py, tests/test_litmus_model.py): numpy slice
 * assignment, np.add.at / np.bincount, np.sum, math.fsum, np.concatenate,
 * reshape/transpose closed forms, hand-computed 2-PE programs, and a brute-force
 * schedule enumerator that is independent of this file.
 * Parity against values printed in the paper: UNPINNED -- the paper prints no
 * numeric example (L510); only its ordering/visibility rules are pinned.
 *
 * State: heap[p] = heap + p*heap_bytes, p = 0..npes-1 ("symmetric heap ... exists
 * at each PE with the same size and allocation order", L108-L114).  All operands
 * are symmetric offsets (L202, L355); AMO values are immediates.
 */
#include <stdint.h>
#include <string.h>

/* opcodes of the oracle's own descriptor format */
enum {
    ORC_PUT = 1, ORC_GET = 2, ORC_PUT_SIGNAL = 3, ORC_ATOMIC_ADD = 4, ORC_ATOMIC_FETCH_ADD = 5,
    ORC_ATOMIC_COMPARE_SWAP = 6, ORC_SIGNAL_WAIT_UNTIL = 7, ORC_FENCE = 8, ORC_QUIET = 9,
    ORC_BARRIER_ALL = 10
};
enum { ORC_SIGNAL_SET = 0, ORC_SIGNAL_ADD = 1 };
enum { ORC_CMP_EQ = 0, ORC_CMP_NE, ORC_CMP_GT, ORC_CMP_GE, ORC_CMP_LT, ORC_CMP_LE };
enum { ORC_OK = 0, ORC_ERR_RANGE = 1, ORC_ERR_WAIT_UNSATISFIED = 2, ORC_ERR_OPCODE = 3, ORC_ERR_ALIGN = 4 };

typedef struct {
    int32_t opcode, initiator, target, sig_op, cmp, _pad;
    uint64_t rem_off;   /* offset in the TARGET's heap   (put dest, get source, AMO word)        */
    uint64_t loc_off;   /* offset in the INITIATOR's heap (put source, get dest, fetch, wait word) */
    uint64_t nbytes;
    uint64_t value;     /* AMO operand / signal value / wait comparand */
    uint64_t cond;      /* compare-swap condition */
    uint64_t sig_off;   /* signal word in the TARGET's heap (put_signal) */
} orc_op_t;

static uint64_t ld64(const uint8_t *p) { uint64_t v; memcpy(&v, p, 8); return v; }
static void st64(uint8_t *p, uint64_t v) { memcpy(p, &v, 8); }

static int in_range(uint64_t off, uint64_t n, uint64_t heap_bytes) {
    return off <= heap_bytes && n <= heap_bytes - off;
}

/*
 * Execute ops[0..nops) in index order.  Returns ORC_OK or an error code with the
 * offending op index in *err_index.  SURVEY.md 8(c) table, row by row.
 */
int orc_exec_batch(uint8_t *heap, int npes, uint64_t heap_bytes, const orc_op_t *ops, uint64_t nops,
                   uint64_t *err_index) {
    for (uint64_t k = 0; k < nops; ++k) {
        const orc_op_t *o = &ops[k];
        *err_index = k;
        if (o->opcode == ORC_FENCE || o->opcode == ORC_QUIET || o->opcode == ORC_BARRIER_ALL) {
            /* L377: "A fence orders subsequent operations with respect to prior ones ... quiet ensures
             * completion of outstanding operations initiated by the caller"; L369 barrier is a visibility
             * point.  In this schedule every earlier op has already completed: nothing to do. */
            continue;
        }
        if (o->initiator < 0 || o->initiator >= npes || o->target < 0 || o->target >= npes) return ORC_ERR_RANGE;
        uint8_t *ini = heap + (uint64_t)o->initiator * heap_bytes;
        uint8_t *tgt = heap + (uint64_t)o->target * heap_bytes;
        switch (o->opcode) {
        case ORC_PUT:            /* "A put updates remote memory" (L116) */
        case ORC_PUT_SIGNAL:
            if (!in_range(o->rem_off, o->nbytes, heap_bytes) || !in_range(o->loc_off, o->nbytes, heap_bytes))
                return ORC_ERR_RANGE;
            memmove(tgt + o->rem_off, ini + o->loc_off, o->nbytes);
            if (o->opcode == ORC_PUT_SIGNAL) {
                /* put-with-signal (L218, L461): the signal word in the target's heap is updated after
                 * the payload; SET or ADD (SURVEY.md reading 8). */
                if (!in_range(o->sig_off, 8, heap_bytes)) return ORC_ERR_RANGE;
                if (o->sig_off & 7) return ORC_ERR_ALIGN;
                if (o->sig_op == ORC_SIGNAL_SET) st64(tgt + o->sig_off, o->value);
                else st64(tgt + o->sig_off, ld64(tgt + o->sig_off) + o->value);
            }
            break;
        case ORC_GET:            /* "a get fetches remote data into local memory" (L116) */
            if (!in_range(o->rem_off, o->nbytes, heap_bytes) || !in_range(o->loc_off, o->nbytes, heap_bytes))
                return ORC_ERR_RANGE;
            memmove(ini + o->loc_off, tgt + o->rem_off, o->nbytes);
            break;
        case ORC_ATOMIC_ADD: {   /* "combine remote update with a compute operation (e.g., atomic add)" (L116) */
            if (!in_range(o->rem_off, 8, heap_bytes)) return ORC_ERR_RANGE;
            if (o->rem_off & 7) return ORC_ERR_ALIGN;
            st64(tgt + o->rem_off, ld64(tgt + o->rem_off) + o->value);     /* mod 2^64 */
            break;
        }
        case ORC_ATOMIC_FETCH_ADD: {   /* "may return the value prior to the update" (L116) */
            if (!in_range(o->rem_off, 8, heap_bytes) || !in_range(o->loc_off, 8, heap_bytes)) return ORC_ERR_RANGE;
            if ((o->rem_off | o->loc_off) & 7) return ORC_ERR_ALIGN;
            uint64_t old = ld64(tgt + o->rem_off);
            st64(tgt + o->rem_off, old + o->value);
            st64(ini + o->loc_off, old);
            break;
        }
        case ORC_ATOMIC_COMPARE_SWAP: {   /* OpenSHMEM 1.6 compare-swap, inherited via L361/L363 */
            if (!in_range(o->rem_off, 8, heap_bytes) || !in_range(o->loc_off, 8, heap_bytes)) return ORC_ERR_RANGE;
            if ((o->rem_off | o->loc_off) & 7) return ORC_ERR_ALIGN;
            uint64_t old = ld64(tgt + o->rem_off);
            if (old == o->cond) st64(tgt + o->rem_off, o->value);
            st64(ini + o->loc_off, old);
            break;
        }
        case ORC_SIGNAL_WAIT_UNTIL: {   /* wait (L116, L392): unsigned 64-bit comparison, reading 9 */
            if (!in_range(o->loc_off, 8, heap_bytes)) return ORC_ERR_RANGE;
            if (o->loc_off & 7) return ORC_ERR_ALIGN;
            uint64_t s = ld64(ini + o->loc_off), v = o->value;
            int ok;
            switch (o->cmp) {
            case ORC_CMP_EQ: ok = (s == v); break;
            case ORC_CMP_NE: ok = (s != v); break;
            case ORC_CMP_GT: ok = (s > v); break;
            case ORC_CMP_GE: ok = (s >= v); break;
            case ORC_CMP_LT: ok = (s < v); break;
            case ORC_CMP_LE: ok = (s <= v); break;
            default: return ORC_ERR_OPCODE;
            }
            /* batch index order must be a valid sequential schedule */
            if (!ok) return ORC_ERR_WAIT_UNSATISFIED;
            break;
        }
        default:
            return ORC_ERR_OPCODE;
        }
    }
    *err_index = nops;
    return ORC_OK;
}

/* ---- homogeneous AMO batches (structure-of-arrays), executed in index order ------------------
 * Word k of the symmetric int64/uint64 array at sym_off on PE tgt_pe[i] is
 * heap[tgt_pe[i]][sym_off + 8*idx[i]].  Values are immediates (L355). */

int orc_atomic_add_batch(uint8_t *heap, int npes, uint64_t heap_bytes, uint64_t sym_off,
                         const int32_t *tgt_pe, const uint64_t *idx, const uint64_t *val, uint64_t n) {
    for (uint64_t i = 0; i < n; ++i) {
        uint64_t off = sym_off + 8 * idx[i];
        if (tgt_pe[i] < 0 || tgt_pe[i] >= npes || !in_range(off, 8, heap_bytes)) return ORC_ERR_RANGE;
        uint8_t *w = heap + (uint64_t)tgt_pe[i] * heap_bytes + off;
        st64(w, ld64(w) + val[i]);
    }
    return ORC_OK;
}

int orc_atomic_fetch_add_batch(uint8_t *heap, int npes, uint64_t heap_bytes, uint64_t sym_off,
                               const int32_t *tgt_pe, const uint64_t *idx, const uint64_t *val,
                               uint64_t *fetched, uint64_t n) {
    for (uint64_t i = 0; i < n; ++i) {
        uint64_t off = sym_off + 8 * idx[i];
        if (tgt_pe[i] < 0 || tgt_pe[i] >= npes || !in_range(off, 8, heap_bytes)) return ORC_ERR_RANGE;
        uint8_t *w = heap + (uint64_t)tgt_pe[i] * heap_bytes + off;
        uint64_t old = ld64(w);
        st64(w, old + val[i]);
        fetched[i] = old;
    }
    return ORC_OK;
}

int orc_atomic_compare_swap_batch(uint8_t *heap, int npes, uint64_t heap_bytes, uint64_t sym_off,
                                  const int32_t *tgt_pe, const uint64_t *idx, const uint64_t *cond,
                                  const uint64_t *val, uint64_t *fetched, uint64_t n) {
    for (uint64_t i = 0; i < n; ++i) {
        uint64_t off = sym_off + 8 * idx[i];
        if (tgt_pe[i] < 0 || tgt_pe[i] >= npes || !in_range(off, 8, heap_bytes)) return ORC_ERR_RANGE;
        uint8_t *w = heap + (uint64_t)tgt_pe[i] * heap_bytes + off;
        uint64_t old = ld64(w);
        if (old == cond[i]) st64(w, val[i]);
        fetched[i] = old;
    }
    return ORC_OK;
}

/* ---- collectives on the world team (each is one atomic unit in batch order) ---- */

/* sum_reduce, fp32: r[k] = sum over p (ascending PE order) of heap[p][src+4k], accumulated in fp64,
 * rounded to nearest fp32 once; every PE's dest receives r (all-reduce; readings 13, 14).  L226. */
int orc_sum_reduce_f32(uint8_t *heap, int npes, uint64_t heap_bytes, uint64_t dst_off, uint64_t src_off,
                       uint64_t nreduce, double *r64_out /* optional: the fp64 sums, may be NULL */) {
    if (!in_range(src_off, 4 * nreduce, heap_bytes) || !in_range(dst_off, 4 * nreduce, heap_bytes)) return ORC_ERR_RANGE;
    for (uint64_t k = 0; k < nreduce; ++k) {
        double acc = 0.0;
        for (int p = 0; p < npes; ++p) {
            float x; memcpy(&x, heap + (uint64_t)p * heap_bytes + src_off + 4 * k, 4);
            acc += (double)x;
        }
        if (r64_out) r64_out[k] = acc;
        float r = (float)acc;
        for (int p = 0; p < npes; ++p) memcpy(heap + (uint64_t)p * heap_bytes + dst_off + 4 * k, &r, 4);
    }
    return ORC_OK;
}

/* sum_reduce, int64: wraparound two's-complement sum (bit-exact). */
int orc_sum_reduce_i64(uint8_t *heap, int npes, uint64_t heap_bytes, uint64_t dst_off, uint64_t src_off,
                       uint64_t nreduce) {
    if (!in_range(src_off, 8 * nreduce, heap_bytes) || !in_range(dst_off, 8 * nreduce, heap_bytes)) return ORC_ERR_RANGE;
    for (uint64_t k = 0; k < nreduce; ++k) {
        uint64_t acc = 0;
        for (int p = 0; p < npes; ++p) acc += ld64(heap + (uint64_t)p * heap_bytes + src_off + 8 * k);
        for (int p = 0; p < npes; ++p) st64(heap + (uint64_t)p * heap_bytes + dst_off + 8 * k, acc);
    }
    return ORC_OK;
}

/* fcollect: for all j, p: heap[j][dst + p*n : +n] = heap[p][src : +n]  (concatenation in PE order) */
int orc_fcollect(uint8_t *heap, int npes, uint64_t heap_bytes, uint64_t dst_off, uint64_t src_off, uint64_t n) {
    if (!in_range(src_off, n, heap_bytes) || !in_range(dst_off, n * (uint64_t)npes, heap_bytes)) return ORC_ERR_RANGE;
    for (int j = 0; j < npes; ++j)
        for (int p = 0; p < npes; ++p)
            memcpy(heap + (uint64_t)j * heap_bytes + dst_off + (uint64_t)p * n,
                   heap + (uint64_t)p * heap_bytes + src_off, n);
    return ORC_OK;
}

/* alltoall: for all i, j: heap[j][dst + i*n : +n] = heap[i][src + j*n : +n]; src and dst ranges must
 * not overlap (reading 12), so reading the live heap equals reading a snapshot.  L218, L68. */
int orc_alltoall(uint8_t *heap, int npes, uint64_t heap_bytes, uint64_t dst_off, uint64_t src_off, uint64_t n) {
    uint64_t tot = n * (uint64_t)npes;
    if (!in_range(src_off, tot, heap_bytes) || !in_range(dst_off, tot, heap_bytes)) return ORC_ERR_RANGE;
    if (!(src_off + tot <= dst_off || dst_off + tot <= src_off)) return ORC_ERR_RANGE;
    for (int i = 0; i < npes; ++i)
        for (int j = 0; j < npes; ++j)
            memcpy(heap + (uint64_t)j * heap_bytes + dst_off + (uint64_t)i * n,
                   heap + (uint64_t)i * heap_bytes + src_off + (uint64_t)j * n, n);
    return ORC_OK;
}

/* block-strided alltoall (the transpose of "FFT-driven spectral phases, many-to-many exchanges",
 * L68; generalises OpenSHMEM 1.6 alltoalls, inherited via L361): for all source PEs i, destination PEs j and blocks b < nblocks
 *     heap[j][dst + i*dst_pe_stride + b*dst_block_stride : +block] = heap[i][src + j*src_pe_stride + b*src_block_stride : +block]
 * (strides in bytes).  alltoalls(dest, source, dst, sst, nelems) on elements of es bytes is the case block = es, nblocks = nelems,
 * block strides = dst*es / sst*es, pe strides = nelems*dst*es / nelems*sst*es.  Source and destination footprints must not
 * overlap, and no two (i, b) may write the same destination bytes (both undefined otherwise). */
int orc_alltoalls(uint8_t *heap, int npes, uint64_t heap_bytes, uint64_t dst_off, uint64_t src_off, uint64_t dst_pe_stride,
                  uint64_t src_pe_stride, uint64_t dst_block_stride, uint64_t src_block_stride, uint64_t block,
                  uint64_t nblocks) {
    if (block == 0 || nblocks == 0) return ORC_OK;
    uint64_t dspan = (uint64_t)(npes - 1) * dst_pe_stride + (nblocks - 1) * dst_block_stride + block;
    uint64_t sspan = (uint64_t)(npes - 1) * src_pe_stride + (nblocks - 1) * src_block_stride + block;
    if (!in_range(dst_off, dspan, heap_bytes) || !in_range(src_off, sspan, heap_bytes)) return ORC_ERR_RANGE;
    if (!(src_off + sspan <= dst_off || dst_off + dspan <= src_off)) return ORC_ERR_RANGE;
    for (int i = 0; i < npes; ++i)
        for (int j = 0; j < npes; ++j)
            for (uint64_t b = 0; b < nblocks; ++b)
                memcpy(heap + (uint64_t)j * heap_bytes + dst_off + (uint64_t)i * dst_pe_stride + b * dst_block_stride,
                       heap + (uint64_t)i * heap_bytes + src_off + (uint64_t)j * src_pe_stride + b * src_block_stride, block);
    return ORC_OK;
}

/* Two-space model (L313-L317, Fig. 4: "CPU space: default symmetric heap (host-attached)" beside the GPU space): a put / get
 * whose operands may live in either space.  The two spaces are two independent arrays of npes windows; `dheap` / `sheap` are the
 * destination's and the source's space.  put: heap_dst[target][dst : +n] = heap_src[pe][src : +n]; get: heap_dst[pe][dst : +n] =
 * heap_src[target][src : +n] -- the caller passes (dst_pe, src_pe) accordingly. */
int orc_copy_spaces(uint8_t *dheap, uint64_t dheap_bytes, uint8_t *sheap, uint64_t sheap_bytes, int npes, int dst_pe, uint64_t dst_off,
                    int src_pe, uint64_t src_off, uint64_t n) {
    if (dst_pe < 0 || dst_pe >= npes || src_pe < 0 || src_pe >= npes) return ORC_ERR_RANGE;
    if (!in_range(dst_off, n, dheap_bytes) || !in_range(src_off, n, sheap_bytes)) return ORC_ERR_RANGE;
    memmove(dheap + (uint64_t)dst_pe * dheap_bytes + dst_off, sheap + (uint64_t)src_pe * sheap_bytes + src_off, n);
    return ORC_OK;
}

/* ---- the rest of the OpenSHMEM op surface on the same heaps --------------
 * The paper names these only by reference: broadcast among the host-side _on_stream variants (L218),
 * "quiet, wait, and test" (L392), the AMO set and strided transfers through "inherited unchanged from
 * OpenSHMEM 1.6" (L361).  Each is its plain definition, executed sequentially. */

/* broadcast (team-based form): for all j (root included): heap[j][dst : +n] = heap[root][src : +n].  L218. */
int orc_broadcast(uint8_t *heap, int npes, uint64_t heap_bytes, uint64_t dst_off, uint64_t src_off, uint64_t n,
                  int root) {
    if (root < 0 || root >= npes) return ORC_ERR_RANGE;
    if (!in_range(src_off, n, heap_bytes) || !in_range(dst_off, n, heap_bytes)) return ORC_ERR_RANGE;
    if (!(src_off + n <= dst_off || dst_off + n <= src_off)) return ORC_ERR_RANGE;
    for (int j = 0; j < npes; ++j)
        memcpy(heap + (uint64_t)j * heap_bytes + dst_off, heap + (uint64_t)root * heap_bytes + src_off, n);
    return ORC_OK;
}

/* reductions: every PE's dest[k] = op over p (ASCENDING PE order) of source[k] on PE p (all-reduce).
 * dtypes: 0 = fp32 (sum / prod accumulated in fp64, rounded to fp32 once; min / max exact),
 *         1 = int64, 2 = int32 (wraparound two's-complement sum / prod; signed min / max; bitwise),
 *         3 = fp64 (sum / prod accumulated in fp64 in PE order; min / max exact).
 * Inputs of the floating-point reductions are NaN-free (undefined otherwise). */
enum { ORC_RED_SUM = 0, ORC_RED_PROD, ORC_RED_MIN, ORC_RED_MAX, ORC_RED_AND, ORC_RED_OR, ORC_RED_XOR };
enum { ORC_T_F32 = 0, ORC_T_I64 = 1, ORC_T_I32 = 2, ORC_T_F64 = 3 };

static double red_f(int op, double a, double b) {
    switch (op) {
    case ORC_RED_SUM: return a + b;
    case ORC_RED_PROD: return a * b;
    case ORC_RED_MIN: return b < a ? b : a;
    default: return b > a ? b : a;
    }
}
static uint64_t red_u(int op, uint64_t a, uint64_t b, int is32) {
    switch (op) {
    case ORC_RED_SUM: return a + b;
    case ORC_RED_PROD: return a * b;
    case ORC_RED_MIN: return is32 ? ((int32_t)b < (int32_t)a ? b : a) : ((int64_t)b < (int64_t)a ? b : a);
    case ORC_RED_MAX: return is32 ? ((int32_t)b > (int32_t)a ? b : a) : ((int64_t)b > (int64_t)a ? b : a);
    case ORC_RED_AND: return a & b;
    case ORC_RED_OR: return a | b;
    default: return a ^ b;
    }
}

int orc_reduce(uint8_t *heap, int npes, uint64_t heap_bytes, int op, int dtype, uint64_t dst_off, uint64_t src_off,
               uint64_t nreduce) {
    const uint64_t es = (dtype == ORC_T_I64 || dtype == ORC_T_F64) ? 8 : 4;
    if (op < ORC_RED_SUM || op > ORC_RED_XOR || dtype < ORC_T_F32 || dtype > ORC_T_F64) return ORC_ERR_OPCODE;
    if ((dtype == ORC_T_F32 || dtype == ORC_T_F64) && op >= ORC_RED_AND) return ORC_ERR_OPCODE;
    if (!in_range(src_off, es * nreduce, heap_bytes) || !in_range(dst_off, es * nreduce, heap_bytes)) return ORC_ERR_RANGE;
    for (uint64_t k = 0; k < nreduce; ++k) {
        uint8_t out[8];
        if (dtype == ORC_T_F32 || dtype == ORC_T_F64) {
            double acc = 0.0;
            for (int p = 0; p < npes; ++p) {
                const uint8_t *q = heap + (uint64_t)p * heap_bytes + src_off + es * k;
                double x;
                if (dtype == ORC_T_F32) { float f; memcpy(&f, q, 4); x = (double)f; } else memcpy(&x, q, 8);
                acc = p == 0 ? (op == ORC_RED_SUM ? 0.0 + x : x) : red_f(op, acc, x);   /* SUM starts from +0.0, as orc_sum_reduce_f32 */
            }
            if (dtype == ORC_T_F32) { float f = (float)acc; memcpy(out, &f, 4); } else memcpy(out, &acc, 8);
        } else {
            uint64_t acc = 0;
            for (int p = 0; p < npes; ++p) {
                const uint8_t *q = heap + (uint64_t)p * heap_bytes + src_off + es * k;
                uint64_t x = 0;
                memcpy(&x, q, es);
                acc = p == 0 ? x : red_u(op, acc, x, es == 4);
            }
            memcpy(out, &acc, es);          /* little-endian: the low `es` bytes */
        }
        for (int p = 0; p < npes; ++p) memcpy(heap + (uint64_t)p * heap_bytes + dst_off + es * k, out, es);
    }
    return ORC_OK;
}

/* generic AMO batch, structure-of-arrays, executed in index order on `width`-byte words (4 or 8):
 *   word = heap[tgt_pe[i]][sym_off + width*idx[i]];  old = word;  word = f(old, val[i]);  fetched[i] = old (if asked).
 * ADD / AND / OR / XOR; SWAP (word = val; without `fetched` this is atomic_set); FETCH (word unchanged: atomic_fetch).
 * inc / fetch_inc are ADD with val = 1.  (OpenSHMEM 1.6 AMO set, L361.) */
enum { ORC_AMO_ADD = 0, ORC_AMO_AND, ORC_AMO_OR, ORC_AMO_XOR, ORC_AMO_SWAP, ORC_AMO_FETCH };

int orc_amo_batch(uint8_t *heap, int npes, uint64_t heap_bytes, int op, int width, uint64_t sym_off,
                  const int32_t *tgt_pe, const uint64_t *idx, const uint64_t *val, uint64_t *fetched, uint64_t n) {
    if (op < ORC_AMO_ADD || op > ORC_AMO_FETCH || (width != 4 && width != 8)) return ORC_ERR_OPCODE;
    if (sym_off % (uint64_t)width) return ORC_ERR_ALIGN;
    const uint64_t mask = width == 8 ? ~0ull : 0xffffffffull;
    for (uint64_t i = 0; i < n; ++i) {
        if (tgt_pe[i] < 0 || tgt_pe[i] >= npes || !in_range(sym_off + (uint64_t)width * idx[i], (uint64_t)width, heap_bytes))
            return ORC_ERR_RANGE;
        uint8_t *w = heap + (uint64_t)tgt_pe[i] * heap_bytes + sym_off + (uint64_t)width * idx[i];
        uint64_t old = 0, v = val ? (val[i] & mask) : 0, nw;
        memcpy(&old, w, (size_t)width);
        switch (op) {
        case ORC_AMO_ADD: nw = old + v; break;
        case ORC_AMO_AND: nw = old & v; break;
        case ORC_AMO_OR: nw = old | v; break;
        case ORC_AMO_XOR: nw = old ^ v; break;
        case ORC_AMO_SWAP: nw = v; break;
        default: nw = old; break;
        }
        nw &= mask;
        memcpy(w, &nw, (size_t)width);
        if (fetched) fetched[i] = old;
    }
    return ORC_OK;
}

/* compare-swap batch on `width`-byte words (4 or 8), structure-of-arrays, executed in index order (the compare_swap of the
 * OpenSHMEM 1.6 AMO set on its 32- and 64-bit types, inherited unchanged: L361, L363):
 *   word = heap[tgt_pe[i]][sym_off + width*idx[i]];  old = word;  if (old == cond[i]) word = val[i];  fetched[i] = old.
 * cond and val are taken modulo 2^(8*width); fetched is zero-extended. */
int orc_amo_cswap_batch(uint8_t *heap, int npes, uint64_t heap_bytes, int width, uint64_t sym_off, const int32_t *tgt_pe,
                        const uint64_t *idx, const uint64_t *cond, const uint64_t *val, uint64_t *fetched, uint64_t n) {
    if (width != 4 && width != 8) return ORC_ERR_OPCODE;
    if (sym_off % (uint64_t)width) return ORC_ERR_ALIGN;
    const uint64_t mask = width == 8 ? ~0ull : 0xffffffffull;
    for (uint64_t i = 0; i < n; ++i) {
        if (tgt_pe[i] < 0 || tgt_pe[i] >= npes || !in_range(sym_off + (uint64_t)width * idx[i], (uint64_t)width, heap_bytes))
            return ORC_ERR_RANGE;
        uint8_t *w = heap + (uint64_t)tgt_pe[i] * heap_bytes + sym_off + (uint64_t)width * idx[i];
        uint64_t old = 0;
        memcpy(&old, w, (size_t)width);
        if (old == (cond[i] & mask)) {
            const uint64_t nw = val[i] & mask;
            memcpy(w, &nw, (size_t)width);
        }
        fetched[i] = old;
    }
    return ORC_OK;
}

/* block-strided put / get (OpenSHMEM 1.6 ibput / ibget; iput / iget are the case block = one element):
 * for b in [0, nblocks): dest[b*dst_stride : +block] = source[b*src_stride : +block], strides in BYTES.
 * put: source on `pe`, dest on `target`; get: source on `target`, dest on `pe`. */
int orc_ibput(uint8_t *heap, int npes, uint64_t heap_bytes, uint64_t dst_off, uint64_t src_off, uint64_t dst_stride,
              uint64_t src_stride, uint64_t block, uint64_t nblocks, int pe, int target, int is_get) {
    if (pe < 0 || pe >= npes || target < 0 || target >= npes) return ORC_ERR_RANGE;
    if (nblocks == 0 || block == 0) return ORC_OK;
    if (!in_range(dst_off, (nblocks - 1) * dst_stride + block, heap_bytes) ||
        !in_range(src_off, (nblocks - 1) * src_stride + block, heap_bytes)) return ORC_ERR_RANGE;
    const int dpe = is_get ? pe : target, spe = is_get ? target : pe;
    for (uint64_t b = 0; b < nblocks; ++b)
        memmove(heap + (uint64_t)dpe * heap_bytes + dst_off + b * dst_stride,
                heap + (uint64_t)spe * heap_bytes + src_off + b * src_stride, block);
    return ORC_OK;
}

/* signal test (L392): 1 if cmp(heap[pe][sig_off] as u64, value) holds now, else 0; never blocks. */
int orc_signal_test(const uint8_t *heap, int npes, uint64_t heap_bytes, uint64_t sig_off, int cmp, uint64_t value,
                    int pe) {
    if (pe < 0 || pe >= npes || !in_range(sig_off, 8, heap_bytes) || (sig_off & 7)) return -1;
    const uint64_t s = ld64(heap + (uint64_t)pe * heap_bytes + sig_off);
    switch (cmp) {
    case ORC_CMP_EQ: return s == value;
    case ORC_CMP_NE: return s != value;
    case ORC_CMP_GT: return s > value;
    case ORC_CMP_GE: return s >= value;
    case ORC_CMP_LT: return s < value;
    case ORC_CMP_LE: return s <= value;
    default: return -1;
    }
}

/* vector forms of test (OpenSHMEM 1.6 test_all / test_any / test_some on nelems consecutive u64 words; L392): evaluated on
 * the current state, never block.  `indices` (may be NULL) receives the satisfied positions in ascending order; the return
 * value is their number, or -1 on a bad argument.  all: count == nelems; any: count > 0, the reported index is indices[0]
 * (the LOWEST satisfied position); some: the whole list.  The wait_until_* forms are the same predicates required to hold
 * (in a sequential schedule a wait must already be satisfied at its turn). */
int64_t orc_signal_test_vec(const uint8_t *heap, int npes, uint64_t heap_bytes, uint64_t sig_off, uint64_t nelems, int cmp,
                            uint64_t value, int pe, uint64_t *indices) {
    if (pe < 0 || pe >= npes || (sig_off & 7) || !in_range(sig_off, 8 * nelems, heap_bytes)) return -1;
    int64_t cnt = 0;
    for (uint64_t k = 0; k < nelems; ++k) {
        const int r = orc_signal_test(heap, npes, heap_bytes, sig_off + 8 * k, cmp, value, pe);
        if (r < 0) return -1;
        if (r) { if (indices) indices[cnt] = k; ++cnt; }
    }
    return cnt;
}

/* ---- team collectives ("PE collectives remain collective over a team of
 * PEs").  A team is the strided PE set { start + k*stride : 0 <= k < size } (shmem_team_split_strided); team rank k is that
 * PE.  Each collective is the world definition with "all PEs" replaced by "all team members, in team-rank order"; heaps of
 * PEs outside the team are untouched.  The root of a broadcast is a TEAM RANK. */
static int team_ok(int npes, int start, int stride, int size) {
    return size >= 1 && start >= 0 && stride >= 1 && (long long)start + (long long)(size - 1) * stride < npes;
}
#define TPE(k) ((uint64_t)(start + (k) * stride))

int orc_team_fcollect(uint8_t *heap, int npes, uint64_t heap_bytes, int start, int stride, int size, uint64_t dst_off,
                      uint64_t src_off, uint64_t n) {
    if (!team_ok(npes, start, stride, size)) return ORC_ERR_RANGE;
    if (!in_range(src_off, n, heap_bytes) || !in_range(dst_off, n * (uint64_t)size, heap_bytes)) return ORC_ERR_RANGE;
    for (int j = 0; j < size; ++j)
        for (int k = 0; k < size; ++k)
            memcpy(heap + TPE(j) * heap_bytes + dst_off + (uint64_t)k * n, heap + TPE(k) * heap_bytes + src_off, n);
    return ORC_OK;
}

int orc_team_alltoall(uint8_t *heap, int npes, uint64_t heap_bytes, int start, int stride, int size, uint64_t dst_off,
                      uint64_t src_off, uint64_t n) {
    const uint64_t tot = n * (uint64_t)size;
    if (!team_ok(npes, start, stride, size)) return ORC_ERR_RANGE;
    if (!in_range(src_off, tot, heap_bytes) || !in_range(dst_off, tot, heap_bytes)) return ORC_ERR_RANGE;
    if (!(src_off + tot <= dst_off || dst_off + tot <= src_off)) return ORC_ERR_RANGE;
    for (int i = 0; i < size; ++i)
        for (int j = 0; j < size; ++j)
            memcpy(heap + TPE(j) * heap_bytes + dst_off + (uint64_t)i * n, heap + TPE(i) * heap_bytes + src_off + (uint64_t)j * n, n);
    return ORC_OK;
}

int orc_team_broadcast(uint8_t *heap, int npes, uint64_t heap_bytes, int start, int stride, int size, uint64_t dst_off,
                       uint64_t src_off, uint64_t n, int root_rank) {
    if (!team_ok(npes, start, stride, size) || root_rank < 0 || root_rank >= size) return ORC_ERR_RANGE;
    if (!in_range(src_off, n, heap_bytes) || !in_range(dst_off, n, heap_bytes)) return ORC_ERR_RANGE;
    if (!(src_off + n <= dst_off || dst_off + n <= src_off)) return ORC_ERR_RANGE;
    for (int j = 0; j < size; ++j)
        memcpy(heap + TPE(j) * heap_bytes + dst_off, heap + TPE(root_rank) * heap_bytes + src_off, n);
    return ORC_OK;
}

/* reduction over the team: gather the members' source rows into a scratch world of `size` PEs, reduce there with
 * orc_reduce (ascending team rank = ascending scratch PE), scatter the result rows back to the members' dest. */
#include <stdlib.h>
int orc_team_reduce(uint8_t *heap, int npes, uint64_t heap_bytes, int start, int stride, int size, int op, int dtype,
                    uint64_t dst_off, uint64_t src_off, uint64_t nreduce) {
    const uint64_t es = (dtype == ORC_T_I64 || dtype == ORC_T_F64) ? 8 : 4, nb = es * nreduce;
    if (!team_ok(npes, start, stride, size)) return ORC_ERR_RANGE;
    if (!in_range(src_off, nb, heap_bytes) || !in_range(dst_off, nb, heap_bytes)) return ORC_ERR_RANGE;
    if (nreduce == 0) return ORC_OK;
    uint8_t *tmp = (uint8_t *)malloc((size_t)size * 2 * nb);
    if (!tmp) return ORC_ERR_RANGE;
    for (int k = 0; k < size; ++k) memcpy(tmp + (uint64_t)k * 2 * nb, heap + TPE(k) * heap_bytes + src_off, nb);
    const int rc = orc_reduce(tmp, size, 2 * nb, op, dtype, nb, 0, nreduce);
    if (rc == ORC_OK)
        for (int k = 0; k < size; ++k) memcpy(heap + TPE(k) * heap_bytes + dst_off, tmp + (uint64_t)k * 2 * nb + nb, nb);
    free(tmp);
    return rc;
}
#undef TPE

/* ---- application-side compute of the halo workload (config C2; SURVEY.md readings 21-23) ------
 * Not part of the specification's operations: the stencil application's own kernels, restated on
 * the CPU so the oracle can run the whole workload.  Both sides implement the same counter-based
 * generator for the perturbation (allowed: "each side implements the same counter-based generator"). */

static uint64_t fin64(uint64_t x) {
    x ^= x >> 30; x *= 0xBF58476D1CE4E5B9ull;
    x ^= x >> 27; x *= 0x94D049BB133111EBull;
    x ^= x >> 31;
    return x;
}
static uint64_t mix64(uint64_t seed, uint64_t stream, uint64_t i) {
    uint64_t x = fin64(seed * 0xD1342543DE82EF95ull + stream * 0x9E3779B97F4A7C15ull + 0x2545F4914F6CDD1Dull);
    return fin64(x ^ (i * 0x9E3779B97F4A7C15ull + 0x632BE59BD9B4E019ull));
}

/* delta(seed, round, gidx) = (mix64 mod 2^16) * 2^-30  (reading 22) */
double orc_halo_delta(uint64_t seed, uint64_t round, uint64_t gidx) {
    return (double)(mix64(seed, round, gidx) & 0xFFFFull) * 0x1.0p-30;
}

/* Perturb PE (px,py,pz)'s B^3 block U (x-major: U[(x*B+y)*B+z]) for one round:
 * U[c] += delta(seed, round, global index of c in the (2B)^3 grid). */
void orc_halo_perturb(double *U, uint64_t B, int px, int py, int pz, uint64_t seed, uint64_t round) {
    uint64_t G = 2 * B;
    for (uint64_t x = 0; x < B; ++x)
        for (uint64_t y = 0; y < B; ++y)
            for (uint64_t z = 0; z < B; ++z) {
                uint64_t g = ((px * B + x) * G + (py * B + y)) * G + (pz * B + z);
                U[(x * B + y) * B + z] += orc_halo_delta(seed, round, g);
            }
}

/* Pack face f = 2*axis + dir (dir 0: index 0, dir 1: index B-1 along axis) of U into send[B*B];
 * the two remaining axes keep their relative order (lower axis major). */
void orc_halo_pack(const double *U, uint64_t B, int f, double *send) {
    int axis = f >> 1, dir = f & 1;
    uint64_t fix = dir ? B - 1 : 0;
    for (uint64_t a = 0; a < B; ++a)
        for (uint64_t b = 0; b < B; ++b) {
            uint64_t x, y, z;
            if (axis == 0)      { x = fix; y = a; z = b; }
            else if (axis == 1) { x = a; y = fix; z = b; }
            else                { x = a; y = b; z = fix; }
            send[a * B + b] = U[(x * B + y) * B + z];
        }
}

/* order-independent checksum of n 64-bit words: sum bits(x_k)*(2k+1) mod 2^64 (reading 23) */
uint64_t orc_checksum64(const uint8_t *p, uint64_t n) {
    uint64_t s = 0;
    for (uint64_t k = 0; k < n; ++k) s += ld64(p + 8 * k) * (2 * k + 1);
    return s;
}
