"""Pins of the NEXT-2 part of the CPU oracle (broadcast, general reductions, generic AMOs, block-strided put/get,
signal test) against things other than itself: numpy library routines (np.tile, ufunc.reduce, ufunc.at, strided slice
assignment, math.fsum / math.prod), hand-computed small cases with the expected heaps written out, and algebraic
identities (a SWAP chain permutes values, XOR twice restores, MIN <= every input).  CPU only."""
import math

import numpy as np
import pytest

from oracle import oracle as orc
from workloads import gen

M64 = (1 << 64) - 1


def world(npes, words, seed, dtype=np.uint64):
    w = orc.OracleWorld(npes, 4 * words * 8 + 1024)
    a, b = w.malloc(words * 8), w.malloc(words * 8)
    init = gen.u64(npes * words, seed).reshape(npes, words)
    w.view(a, words * 8, np.uint64)[:] = init
    return w, a, b, init


# ---- broadcast -------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("root", [0, 3, 6])
def test_broadcast_equals_tile_of_root_row(root):
    w, a, b, init = world(7, 33, 201)
    w.broadcast(b + 3, a + 5, 33 * 8 - 9, root)                     # odd offsets and size
    exp = np.tile(init.view(np.uint8)[root, 5:5 + 33 * 8 - 9], (7, 1))
    assert np.array_equal(w.view(b, 33 * 8)[:, 3:3 + 33 * 8 - 9], exp)
    assert np.array_equal(w.view(a, 33 * 8, np.uint64), init)       # sources untouched
    assert not w.view(b, 33 * 8)[:, :3].any() and not w.view(b, 33 * 8)[:, -6:].any()


def test_broadcast_hand_case_and_errors():
    w = orc.OracleWorld(3, 64)
    w.heap[:, :4] = [[1, 2, 3, 4], [5, 6, 7, 8], [9, 10, 11, 12]]
    w.broadcast(8, 1, 2, 1)
    assert w.heap[:, 8:10].tolist() == [[6, 7]] * 3
    with pytest.raises(orc.OracleError):
        w.broadcast(2, 0, 4, 0)                                     # overlapping source / dest
    with pytest.raises(orc.OracleError):
        w.broadcast(8, 0, 4, 3)                                     # root out of range


# ---- reductions --------------------------------------------------------------------------------------------------------
INT_OPS = {"sum": np.add, "prod": np.multiply, "min": np.minimum, "max": np.maximum, "and": np.bitwise_and,
           "or": np.bitwise_or, "xor": np.bitwise_xor}


@pytest.mark.parametrize("op", sorted(INT_OPS))
@pytest.mark.parametrize("dtype,npdt", [("i64", np.int64), ("i32", np.int32)])
def test_integer_reductions_equal_numpy_ufunc_reduce(op, dtype, npdt):
    npes, n = 9, 257
    es = np.dtype(npdt).itemsize
    w = orc.OracleWorld(npes, 4 * n * 8)
    s, d = w.malloc(n * es), w.malloc(n * es)
    src = gen.u64(npes * n, 211).reshape(npes, n).astype(np.uint64).view(np.int64).astype(npdt)   # low bits; signs mixed
    if op in ("min", "max"):
        src[:, ::7] = -src[:, ::7] // 3
    w.view(s, n * es, npdt)[:] = src
    w.reduce(op, dtype, d, s, n)
    with np.errstate(over="ignore"):
        exp = INT_OPS[op].reduce(src, axis=0, dtype=npdt)                       # wraparound for sum / prod
    out = w.view(d, n * es, npdt)
    assert np.array_equal(out, np.tile(exp, (npes, 1)))
    assert np.array_equal(w.view(s, n * es, npdt), src)


def test_integer_reduction_hand_case():
    w = orc.OracleWorld(3, 256)
    w.view(0, 16, np.int64)[:] = [[5, -2], [-7, 3], [6, 1 << 62]]
    for op, exp in (("sum", [4, (1 << 62) + 1]), ("prod", [-210, (-6 * (1 << 62)) % (1 << 64)]), ("min", [-7, -2]),
                    ("max", [6, 1 << 62]), ("and", [5 & -7 & 6, -2 & 3 & (1 << 62)]), ("or", [5 | -7 | 6, -2 | 3 | (1 << 62)]),
                    ("xor", [5 ^ -7 ^ 6, -2 ^ 3 ^ (1 << 62)])):
        w.reduce(op, "i64", 64, 0, 2)
        got = w.view(64, 16, np.uint64)
        assert got.tolist() == [[e % (1 << 64) for e in exp]] * 3, op


@pytest.mark.parametrize("dtype,npdt", [("f32", np.float32), ("f64", np.float64)])
def test_float_reductions(dtype, npdt):
    npes, n = 16, 301
    es = np.dtype(npdt).itemsize
    w = orc.OracleWorld(npes, 4 * n * 8)
    s, d = w.malloc(n * es), w.malloc(n * es)
    src = gen.normal_f32(npes * n, 212).reshape(npes, n).astype(npdt)
    w.view(s, n * es, npdt)[:] = src
    # min / max: exact, equal to numpy's
    for op, uf in (("min", np.minimum), ("max", np.maximum)):
        w.reduce(op, dtype, d, s, n)
        assert np.array_equal(w.view(d, n * es, npdt), np.tile(uf.reduce(src, axis=0), (npes, 1)))
    # sum: the correctly rounded exact sum (math.fsum) within the error bound of an fp64 accumulation
    w.reduce("sum", dtype, d, s, n)
    got = w.view(d, n * es, npdt)
    exact = np.array([math.fsum(src[:, k].astype(np.float64).tolist()) for k in range(n)])
    if npdt == np.float32:
        assert np.array_equal(got[0], exact.astype(np.float32))     # one rounding of an (almost) exact fp64 sum
    else:
        bound = (npes - 1) * 2.0 ** -53 * np.abs(src).sum(axis=0)
        assert (np.abs(got[0] - exact) <= bound).all()
    assert (got == got[0]).all()
    # prod: against math.prod in exact rational arithmetic on a few columns
    from fractions import Fraction
    small = (src[:, :8].astype(np.float64) * 0.5 + 1.0).astype(npdt)           # keep products away from 0 / inf
    w.view(s, n * es, npdt)[:, :8] = small
    w.reduce("prod", dtype, d, s, 8)
    got = w.view(d, n * es, npdt)[0, :8].astype(np.float64)
    for k in range(8):
        exact = math.prod(Fraction(float(x)) for x in small[:, k])
        rel = abs(Fraction(float(got[k])) - exact) / abs(exact)
        assert rel <= (2.0 ** -23 if npdt == np.float32 else npes * 2.0 ** -52)


def test_reduce_rejects_bitwise_on_floats_and_bad_ranges():
    w = orc.OracleWorld(2, 256)
    for op in ("and", "or", "xor"):
        with pytest.raises(orc.OracleError):
            w.reduce(op, "f32", 64, 0, 4)
    with pytest.raises(orc.OracleError):
        w.reduce("sum", "i64", 64, 0, 100)


def test_reduce_sum_agrees_with_the_dedicated_sum_reduce_routines():
    npes, n = 5, 100
    w, a, b, init = world(npes, n, 213)
    w2, a2, b2, _ = world(npes, n, 213)
    w.reduce("sum", "i64", b, a, n)
    w2.sum_reduce_i64(b2, a2, n)
    assert np.array_equal(w.heap, w2.heap)
    f = gen.normal_f32(npes * n, 214).reshape(npes, n)
    w.view(a, n * 4, np.float32)[:] = f
    w2.view(a2, n * 4, np.float32)[:] = f
    w.reduce("sum", "f32", b, a, n)
    w2.sum_reduce_f32(b2, a2, n)
    assert np.array_equal(w.heap, w2.heap)


# ---- generic AMOs ------------------------------------------------------------------------------------------------------
AMO_UFUNC = {"add": np.add, "and": np.bitwise_and, "or": np.bitwise_or, "xor": np.bitwise_xor}


@pytest.mark.parametrize("op", sorted(AMO_UFUNC))
@pytest.mark.parametrize("width,npdt", [(8, np.uint64), (4, np.uint32)])
def test_commutative_amos_equal_ufunc_at(op, width, npdt):
    npes, words, n = 4, 64, 5000
    w = orc.OracleWorld(npes, words * 8 + 512)
    a = w.malloc(words * width)
    init = gen.u64(npes * words, 221).reshape(npes, words).astype(npdt)
    w.view(a, words * width, npdt)[:] = init
    tgt = gen.uniform_i32(n, 0, npes - 1, 222, 0)
    idx = gen.uniform_i32(n, 0, words - 1, 222, 1)
    val = gen.u64(n, 223)
    fetched = w.amo_batch(op, width, a, tgt, idx, val, fetch=True)
    exp = init.copy().reshape(-1)
    flat = tgt.astype(np.int64) * words + idx
    with np.errstate(over="ignore"):
        AMO_UFUNC[op].at(exp, flat, val.astype(npdt))
    assert np.array_equal(w.view(a, words * width, npdt).reshape(-1), exp)
    # fetched values replayed sequentially in index order (independent re-statement with python ints)
    cur = {int(k): int(v) for k, v in enumerate(init.reshape(-1))}
    mask = (1 << (8 * width)) - 1
    pyop = {"add": lambda x, y: (x + y) & mask, "and": lambda x, y: x & y, "or": lambda x, y: x | y, "xor": lambda x, y: x ^ y}[op]
    for i in range(300):
        k = int(flat[i])
        assert int(fetched[i]) == cur[k]
        cur[k] = pyop(cur[k], int(val[i]) & mask)


def test_swap_set_fetch_hand_cases():
    w = orc.OracleWorld(2, 128)
    w.view(0, 32, np.uint64)[:] = [[1, 2, 3, 4], [5, 6, 7, 8]]
    f = w.amo_batch("swap", 8, 0, [1, 1, 0], [2, 2, 0], [70, 71, 9], fetch=True)
    assert f.tolist() == [7, 70, 1]
    assert w.view(0, 32, np.uint64).tolist() == [[9, 2, 3, 4], [5, 6, 71, 8]]
    assert w.amo_batch("swap", 8, 0, [0], [3], [M64]) is None                    # atomic_set: no fetch
    assert w.view(0, 32, np.uint64)[0, 3] == M64
    f = w.amo_batch("fetch", 8, 0, [0, 1], [3, 1], None, fetch=True)               # atomic_fetch: word unchanged
    assert f.tolist() == [M64, 6] and w.view(0, 32, np.uint64).tolist() == [[9, 2, 3, M64], [5, 6, 71, 8]]
    # 32-bit words: value truncated, neighbours untouched
    w.amo_batch("add", 4, 0, [1], [1], [0x1_0000_0003])
    assert w.view(0, 32, np.uint32)[1].tolist()[:3] == [5, 3, 6]
    w.amo_batch("xor", 4, 4, [1, 1], [0, 0], [0xdeadbeef, 0xdeadbeef])          # xor twice restores
    assert w.view(0, 32, np.uint32)[1, 1] == 3
    with pytest.raises(orc.OracleError):
        w.amo_batch("add", 8, 4, [0], [0], [1])                                   # misaligned 64-bit word
    with pytest.raises(orc.OracleError):
        w.amo_batch("add", 8, 0, [2], [0], [1])                                   # PE out of range


def test_cswap_hand_cases_both_widths():
    """compare-swap of the inherited AMO set on 32- and 64-bit words, by hand."""
    w = orc.OracleWorld(2, 128)
    w.view(0, 32, np.uint64)[:] = [[1, 2, 3, 4], [5, 6, 7, 8]]
    f = w.amo_cswap_batch(8, 0, [1, 1, 1, 0], [2, 2, 2, 0], [7, 7, 70, 2], [70, 71, 72, 9])
    assert f.tolist() == [7, 70, 70, 1]                              # 1st swaps, 2nd fails (word is 70), 3rd swaps, 4th fails
    assert w.view(0, 32, np.uint64).tolist() == [[1, 2, 3, 4], [5, 6, 72, 8]]
    # 32-bit: the word is one half of a 64-bit cell; cond / val are truncated; the neighbouring half is untouched
    w.view(0, 32, np.uint32)[0, :4] = [10, 11, 12, 13]
    f = w.amo_cswap_batch(4, 0, [0, 0, 0], [1, 1, 2], [0x5_0000_000b, 11, 13], [0x9_0000_0063, 100, 5])
    assert f.tolist() == [11, 99, 12]                                # cond 0x5_0000_000b == 11 mod 2^32; val -> 99
    assert w.view(0, 32, np.uint32)[0, :4].tolist() == [10, 99, 12, 13]
    with pytest.raises(orc.OracleError):
        w.amo_cswap_batch(4, 2, [0], [0], [0], [0])                   # misaligned 32-bit word
    with pytest.raises(orc.OracleError):
        w.amo_cswap_batch(2, 0, [0], [0], [0], [0])                   # no 16-bit AMOs
    with pytest.raises(orc.OracleError):
        w.amo_cswap_batch(4, 0, [0], [32], [0], [0])                  # beyond the window


@pytest.mark.parametrize("width,npdt,empty", [(8, np.uint64, M64), (4, np.uint32, 0xffffffff)])
def test_cswap_claim_first_op_in_index_order_wins(width, npdt, empty):
    """Closed form for claim-style batches (every op is CAS(empty -> its own value) on slots holding `empty`): executed in
    index order, the FIRST op of a slot wins (np.unique(return_index)), it fetches `empty`, every later op of the slot fetches
    the winner's value.  width 8 must also agree with the SoA compare-swap routine that was written for config 4."""
    npes, words, n = 3, 40, 3000
    w = orc.OracleWorld(npes, words * 8 + 256)
    a = w.malloc(words * width)
    w.view(a, words * width, npdt)[:] = empty
    tgt = gen.uniform_i32(n, 0, npes - 1, 231, 0)
    idx = gen.uniform_i32(n, 0, words - 2, 231, 1)                    # the last word of every PE is never touched
    val = (gen.u64(n, 232) >> np.uint64(40)) + np.uint64(1)           # < 2^24 + 1: never equal to `empty`, fits 32 bits
    f = w.amo_cswap_batch(width, a, tgt, idx, np.full(n, empty, dtype=np.uint64), val)
    flat = tgt.astype(np.int64) * words + idx
    keys, first = np.unique(flat, return_index=True)
    exp = np.full(npes * words, empty, dtype=np.uint64)
    exp[keys] = val[first]
    assert np.array_equal(w.view(a, words * width, npdt).reshape(-1).astype(np.uint64), exp)
    expf = exp[flat].copy()
    expf[first] = empty
    assert np.array_equal(f, expf)
    if width == 8:
        w2 = orc.OracleWorld(npes, words * 8 + 256)
        a2 = w2.malloc(words * 8)
        w2.view(a2, words * 8, np.uint64)[:] = M64
        f2 = w2.atomic_compare_swap_batch(a2, tgt, idx, np.full(n, M64, dtype=np.uint64), val)
        assert np.array_equal(f, f2) and np.array_equal(w.heap, w2.heap)


@pytest.mark.parametrize("width", [4, 8])
def test_cswap_general_conditions_replayed_with_python_ints(width):
    """Arbitrary cond / val on few words with small values, so that many swaps succeed and many fail: replayed op by op."""
    npes, words, n = 2, 6, 4000
    mask = (1 << (8 * width)) - 1
    w = orc.OracleWorld(npes, 256)
    npdt = np.uint32 if width == 4 else np.uint64
    init = (gen.u64(npes * words, 233) % np.uint64(4)).astype(npdt).reshape(npes, words)
    w.view(0, words * width, npdt)[:] = init
    tgt = gen.uniform_i32(n, 0, npes - 1, 234, 0)
    idx = gen.uniform_i32(n, 0, words - 1, 234, 1)
    cond = gen.u64(n, 235) % np.uint64(4) + (gen.u64(n, 236) % np.uint64(2) << np.uint64(32))     # bit 32 set in half of them:
    val = gen.u64(n, 237) % np.uint64(4) + (gen.u64(n, 238) % np.uint64(2) << np.uint64(32))      # ignored on 32-bit words only
    f = w.amo_cswap_batch(width, 0, tgt, idx, cond, val)
    cur = [int(x) for x in init.reshape(-1)]
    swaps = 0
    for i in range(n):
        k = int(tgt[i]) * words + int(idx[i])
        assert int(f[i]) == cur[k]
        if cur[k] == int(cond[i]) & mask:
            cur[k] = int(val[i]) & mask
            swaps += 1
    assert 200 < swaps < n - 200
    assert w.view(0, words * width, npdt).reshape(-1).tolist() == cur


def test_swap_chain_permutes_values():
    """Per word, {fetched values} + {final} = {init} + {swapped-in values} as multisets."""
    npes, words, n = 3, 16, 2000
    w = orc.OracleWorld(npes, words * 8 + 256)
    init = np.arange(1, npes * words + 1, dtype=np.uint64).reshape(npes, words) * np.uint64(1 << 32)
    w.view(0, words * 8, np.uint64)[:] = init
    tgt = gen.uniform_i32(n, 0, npes - 1, 224, 0)
    idx = gen.uniform_i32(n, 0, words - 1, 224, 1)
    val = np.arange(1, n + 1, dtype=np.uint64)
    f = w.amo_batch("swap", 8, 0, tgt, idx, val, fetch=True)
    fin = w.view(0, words * 8, np.uint64).reshape(-1)
    flat = tgt.astype(np.int64) * words + idx
    for k in range(npes * words):
        m = flat == k
        assert sorted(f[m].tolist() + [int(fin[k])]) == sorted(val[m].tolist() + [int(init.reshape(-1)[k])])


# ---- block-strided put / get -----------------------------------------------------------------------------------------
@pytest.mark.parametrize("block,ds,ss,nb", [(8, 8, 2048, 256), (8, 24, 8, 100), (2048, 2048, 65536, 16), (3, 7, 5, 50),
                                            (16, 16, 16, 64), (1, 1, 3, 9)])
def test_ibput_ibget_equal_numpy_strided_assignment(block, ds, ss, nb):
    npes = 3
    span = max(ds, ss) * nb + block + 64
    w = orc.OracleWorld(npes, 2 * span + 1024)
    s, d = w.malloc(span), w.malloc(span)
    pay = gen.u64(npes * ((span + 7) // 8), 231).view(np.uint8).reshape(npes, -1)[:, :span]
    w.view(s, span)[:] = pay
    exp = np.zeros((npes, span), dtype=np.uint8)
    w.ibput(d + 5, s + 3, ds, ss, block, nb, 0, 2)
    for b in range(nb):
        exp[2, 5 + b * ds:5 + b * ds + block] = pay[0, 3 + b * ss:3 + b * ss + block]
    assert np.array_equal(w.view(d, span), exp)
    # the same through numpy's strided views when the blocks do not overlap
    if ds >= block:
        v = np.lib.stride_tricks.as_strided(exp[2, 5:], shape=(nb, block), strides=(ds, 1))
        u = np.lib.stride_tricks.as_strided(pay[0, 3:], shape=(nb, block), strides=(ss, 1))
        assert np.array_equal(v, u)
    w.ibget(d + 1, s + 2, ds, ss, block, nb, 1, 0)                  # PE1.dest <- PE0.source
    for b in range(nb):
        exp[1, 1 + b * ds:1 + b * ds + block] = pay[0, 2 + b * ss:2 + b * ss + block]
    assert np.array_equal(w.view(d, span), exp)


def test_ibput_one_block_is_put_and_face_of_a_cube():
    """block = whole transfer: ibput == put.  A z-face of a B^3 cube is the stride-B gather (what the halo pack does)."""
    B = 12
    w = orc.OracleWorld(2, B ** 3 * 8 + B * B * 8 + 1024)
    U, face = w.malloc(B ** 3 * 8), w.malloc(B * B * 8)
    cube = gen.u64(2 * B ** 3, 232).reshape(2, B, B, B)
    w.view(U, B ** 3 * 8, np.uint64)[:] = cube.reshape(2, -1)
    w.ibput(face, U + (B - 1) * 8, 8, B * 8, 8, B * B, 0, 1)        # z = B-1 face of PE 0 -> PE 1
    assert np.array_equal(w.view(face, B * B * 8, np.uint64)[1].reshape(B, B), cube[0, :, :, B - 1])
    w.ibput(face, U + 3 * B * 8, B * 8, B * B * 8, B * 8, B, 1, 0)  # y = 3 face of PE 1 -> PE 0: B rows of B elements
    assert np.array_equal(w.view(face, B * B * 8, np.uint64)[0].reshape(B, B), cube[1, :, 3, :])
    w.ibput(face, U + 2 * B * B * 8, 0, 0, B * B * 8, 1, 0, 1)      # x = 2 face: one contiguous block
    assert np.array_equal(w.view(face, B * B * 8, np.uint64)[1].reshape(B, B), cube[0, 2])


# ---- signal test -------------------------------------------------------------------------------------------------------
def test_signal_test_truth_table():
    from workloads.spec import CMP_EQ, CMP_GE, CMP_GT, CMP_LE, CMP_LT, CMP_NE
    w = orc.OracleWorld(2, 64)
    w.view(8, 8, np.uint64)[1] = 5
    table = {CMP_EQ: (0, 1, 0), CMP_NE: (1, 0, 1), CMP_GT: (1, 0, 0), CMP_GE: (1, 1, 0), CMP_LT: (0, 0, 1), CMP_LE: (0, 1, 1)}
    for cmp, exp in table.items():
        assert tuple(int(w.signal_test(8, cmp, v, 1)) for v in (4, 5, 6)) == exp
    assert w.signal_test(8, CMP_GT, M64, 1) is False                 # unsigned comparison
    assert w.signal_test(8, CMP_EQ, 0, 0) is True                    # PE 0's word is still 0


def test_sum_of_negative_zeros_is_positive_zero_in_both_sum_routines():
    """SUM = 0 + x_0 + x_1 + ... (IEEE: +0.0 + -0.0 = +0.0); MIN / MAX / PROD keep the sign of zero."""
    w = orc.OracleWorld(3, 256)
    w.view(0, 8, np.float32)[:] = np.float32(-0.0)
    w.reduce("sum", "f32", 64, 0, 2)
    assert w.view(64, 8, np.uint32).tolist() == [[0, 0]] * 3
    w.sum_reduce_f32(128, 0, 2)
    assert w.view(128, 8, np.uint32).tolist() == [[0, 0]] * 3
    w.reduce("max", "f32", 64, 0, 2)
    assert w.view(64, 8, np.uint32).tolist() == [[0x80000000] * 2] * 3
    w.reduce("prod", "f32", 64, 0, 2)                    # (-0)(-0)(-0) = -0
    assert w.view(64, 8, np.uint32).tolist() == [[0x80000000] * 2] * 3


def test_signal_test_vec_equals_numpy_flatnonzero():
    from workloads.spec import CMP_EQ, CMP_GE, CMP_GT, CMP_LE, CMP_LT, CMP_NE
    w = orc.OracleWorld(3, 4096)
    vals = (gen.u64(3 * 100, 241) % np.uint64(7)).reshape(3, 100)
    w.view(256, 800, np.uint64)[:] = vals
    ops = {CMP_EQ: np.equal, CMP_NE: np.not_equal, CMP_GT: np.greater, CMP_GE: np.greater_equal, CMP_LT: np.less, CMP_LE: np.less_equal}
    for cmp, f in ops.items():
        for v in (0, 3, 6, 7):
            for pe in range(3):
                got = w.signal_test_vec(256 + 8 * 5, 90, cmp, v, pe)
                assert np.array_equal(got, np.flatnonzero(f(vals[pe, 5:95], np.uint64(v))))
    assert len(w.signal_test_vec(256, 0, CMP_EQ, 0, 0)) == 0
    with pytest.raises(orc.OracleError):
        w.signal_test_vec(260, 4, CMP_EQ, 0, 0)
    with pytest.raises(orc.OracleError):
        w.signal_test_vec(256, 4, CMP_EQ, 0, 3)
