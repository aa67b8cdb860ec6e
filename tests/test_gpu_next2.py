"""GPU parity of the NEXT-2 surface (broadcast, general reductions, generic AMOs, block-strided put/get, signal test)
against the CPU oracle, through the C-ABI.  Sizes span several tiles and a ragged tail; integer and byte work is
bit-exact; floating-point reductions run in the same order and precision on both sides, so they are bit-exact as well
(and asserted within the derived tolerance first)."""
import numpy as np
import pytest
import torch

from oracle import oracle as orc
from paper_2607_08006_b200 import World
from paper_2607_08006_b200.binding import AMO, CMP, F32, F64, I32, I64, RED, SIGNAL, ShmemgError
from workloads import gen

pytestmark = pytest.mark.gpu
DEV = "cuda:0"
M64 = (1 << 64) - 1


def to_dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).to(DEV)


def pair(npes, heap_bytes):
    return World(npes, heap_bytes, DEV), orc.OracleWorld(npes, heap_bytes)


def fill(w, ow, off, ooff, nbytes, seed):
    pay = gen.u64(w.npes * ((nbytes + 7) // 8), seed).view(np.uint8).reshape(w.npes, -1)[:, :nbytes]
    w.view(off, nbytes).copy_(torch.from_numpy(np.ascontiguousarray(pay)))
    ow.view(ooff, nbytes)[:] = pay
    return pay


# ---- broadcast -------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("npes,nbytes,so,do,root", [
    (16, (1 << 20) + 4096 + 16, 0, 0, 5),          # bulk path, several tiles, ragged 16-byte tail
    (128, 32768, 0, 0, 127),                       # C5-shaped: 128 PEs
    (7, 300001, 3, 5, 0),                          # any alignment: register path
    (3, 1, 1, 0, 2), (4, 15, 0, 1, 1), (2, 0, 0, 0, 0),
])
def test_broadcast_matches_oracle(npes, nbytes, so, do, root):
    span = (nbytes + 64 + 255) // 256 * 256
    w, ow = pair(npes, 2 * span + 4096)
    s, d = w.malloc(span), w.malloc(span)
    os_, od = ow.malloc(span), ow.malloc(span)
    fill(w, ow, s, os_, span, 301)
    w.view(d, span).zero_()
    w.broadcast(d + do, s + so, nbytes, root)
    w.quiet(0)
    ow.broadcast(od + do, os_ + so, nbytes, root)
    assert np.array_equal(w.view(d, span).cpu().numpy(), ow.view(od, span))
    assert np.array_equal(w.view(s, span).cpu().numpy(), ow.view(os_, span))


def test_broadcast_errors():
    w = World(4, 1 << 16, DEV)
    a = w.malloc(4096)
    with pytest.raises(ShmemgError):
        w.broadcast(a + 8, a, 64, 0)               # overlap
    with pytest.raises(ShmemgError):
        w.broadcast(a + 2048, a, 64, 4)            # root out of range
    with pytest.raises(ShmemgError):
        w.broadcast(a + 2048, a, 1 << 20, 0)       # out of the window


# ---- reductions --------------------------------------------------------------------------------------------------------
NP_DT = {F32: np.float32, F64: np.float64, I32: np.int32, I64: np.int64}
ORC_DT = {F32: "f32", F64: "f64", I32: "i32", I64: "i64"}
ORC_OP = {RED.SUM: "sum", RED.PROD: "prod", RED.MIN: "min", RED.MAX: "max", RED.AND: "and", RED.OR: "or", RED.XOR: "xor"}


def reduce_input(dtype, op, npes, n, seed):
    if dtype in (F32, F64):
        x = gen.normal_f32(npes * n, seed).reshape(npes, n).astype(NP_DT[dtype])
        if op == RED.PROD:
            x = (x.astype(np.float64) * 0.25 + 1.0).astype(NP_DT[dtype])       # products stay finite and non-zero
        return x
    return gen.u64(npes * n, seed).reshape(npes, n).view(np.int64).astype(NP_DT[dtype])


@pytest.mark.parametrize("op", list(ORC_OP))
@pytest.mark.parametrize("dtype", [F32, F64, I32, I64])
@pytest.mark.parametrize("npes,n,shift", [(7, 20000 + 3, 0), (33, 1027, 1)])
def test_reduce_matches_oracle(op, dtype, npes, n, shift):
    """shift = 1: offsets one element off 16-byte alignment -> the scalar path alone; shift = 0: bulk body + scalar tail."""
    if dtype in (F32, F64) and op >= RED.AND:
        w = World(2, 4096, DEV)
        a = w.malloc(512)
        with pytest.raises(ShmemgError):
            w.reduce(op, dtype, a + 256, a, 4)
        return
    es = np.dtype(NP_DT[dtype]).itemsize
    nb = (n + 4) * es
    w, ow = pair(npes, 2 * ((nb + 255) // 256 * 256) + 4096)
    s, d = w.malloc(nb), w.malloc(nb)
    os_, od = ow.malloc(nb), ow.malloc(nb)
    x = reduce_input(dtype, op, npes, n, 310 + op)
    w.view(s, nb).zero_(); w.view(d, nb).zero_()
    w.view(s + shift * es, n * es, getattr(torch, np.dtype(NP_DT[dtype]).name)).copy_(torch.from_numpy(x))
    ow.view(os_ + shift * es, n * es, NP_DT[dtype])[:] = x
    w.reduce(op, dtype, d + shift * es, s + shift * es, n)
    w.quiet(0)
    ow.reduce(ORC_OP[op], ORC_DT[dtype], od + shift * es, os_ + shift * es, n)
    g = w.view(d, nb).cpu().numpy()
    o = ow.view(od, nb)
    if dtype in (F32, F64):
        gv, ov = g.view(NP_DT[dtype]).astype(np.float64), o.view(NP_DT[dtype]).astype(np.float64)
        # fp32: one rounding of an fp64 accumulation (north_star: 1e-6 relative); fp64: same order, n*eps bound
        tol = 1e-6 if dtype == F32 else npes * 2.0 ** -52
        assert (np.abs(gv - ov) <= tol * np.abs(ov) + 2.0 ** -36).all()
    assert np.array_equal(g, o)                      # same order, same precision: bit-exact
    assert np.array_equal(w.view(s, nb).cpu().numpy(), ow.view(os_, nb))


def test_reduce_in_place_and_full_c5_shape():
    """dest == source (exact aliasing) and the C5 launch shape: 128 PEs x 4 MiB, MAX on int64, sampled columns."""
    npes, n = 128, 512 * 1024
    w = World(npes, 2 * n * 8 + 4096, DEV)
    s = w.malloc(n * 8)
    x = gen.uniform_i64(npes * n, -(1 << 40), 1 << 40, 320).reshape(npes, n)
    w.view(s, n * 8, torch.int64).copy_(torch.from_numpy(x))
    w.reduce(RED.MAX, I64, s, s, n)
    w.quiet(0)
    g = w.view(s, n * 8, torch.int64).cpu().numpy()
    cols = np.unique(np.concatenate([np.arange(0, 4096), np.arange(n - 4096, n), gen.uniform_i64(4096, 0, n - 1, 321)]))
    ow = orc.OracleWorld(npes, len(cols) * 8 + 256)
    ow.view(0, len(cols) * 8, np.int64)[:] = x[:, cols]
    ow.reduce("max", "i64", 0, 0, len(cols))
    assert np.array_equal(g[:, cols], ow.view(0, len(cols) * 8, np.int64))
    assert (g == g[0]).all() and np.array_equal(g[0], x.max(axis=0))           # property at full size


# ---- generic AMOs ------------------------------------------------------------------------------------------------------
ORC_AMO = {AMO.ADD: "add", AMO.AND: "and", AMO.OR: "or", AMO.XOR: "xor", AMO.SWAP: "swap", AMO.FETCH: "fetch"}
PYOP = {AMO.ADD: lambda x, y, m: (x + y) & m, AMO.AND: lambda x, y, m: x & y, AMO.OR: lambda x, y, m: x | y,
        AMO.XOR: lambda x, y, m: x ^ y}


def amo_case(width, npes, words, n, seed, distinct):
    npdt = np.uint64 if width == 8 else np.uint32
    init = gen.u64(npes * words, seed).astype(npdt).reshape(npes, words)
    if distinct:                                         # every word touched at most once: fetched values are unique too
        flat = np.argsort(gen.u64(npes * words, seed + 1), kind="stable")[:n].astype(np.int64)
    else:
        flat = (gen.u64(n, seed + 1) % np.uint64(npes * words)).astype(np.int64)
        flat[::3] = flat[::3] % 7                        # heavy contention on a few words
    return npdt, init, flat, (flat // words).astype(np.int32), (flat % words), gen.u64(n, seed + 2)


@pytest.mark.parametrize("amo", [AMO.ADD, AMO.AND, AMO.OR, AMO.XOR, AMO.SWAP])
@pytest.mark.parametrize("width", [8, 4])
@pytest.mark.parametrize("fetch", [False, True])
@pytest.mark.parametrize("idx_dtype", [np.int32, np.int64])
def test_generic_amo_conflict_free_is_bit_exact(amo, width, fetch, idx_dtype):
    npes, words, n = 5, 3000, 9001
    npdt, init, flat, tgt, idx, val = amo_case(width, npes, words, n, 330 + amo, distinct=True)
    w, ow = pair(npes, words * 8 + 4096)
    pad, opad = w.malloc(256), ow.malloc(256)
    a, oa = w.malloc(words * width), ow.malloc(words * width)
    w.view(a, words * width).copy_(torch.from_numpy(init.view(np.uint8)))
    ow.view(oa, words * width, npdt)[:] = init
    f = torch.zeros(n, dtype=torch.int64, device=DEV) if fetch else None
    w.atomic_op_batch(amo, width, a, to_dev(tgt), to_dev(idx.astype(idx_dtype)), val=to_dev(val.view(np.int64)), fetched_out=f)
    w.quiet(0)
    of = ow.amo_batch(ORC_AMO[amo], width, oa, tgt, idx, val, fetch=fetch)
    assert np.array_equal(w.view(a, words * width).cpu().numpy(), ow.view(oa, words * width))
    if fetch:
        assert np.array_equal(f.cpu().numpy().view(np.uint64), of)


@pytest.mark.parametrize("amo", [AMO.ADD, AMO.AND, AMO.OR, AMO.XOR])
@pytest.mark.parametrize("width", [8, 4])
def test_generic_amo_contended_commutative_finals_and_fetch_chains(amo, width):
    """Heavy contention.  Final words are schedule independent (commutative ops): bit-exact against the oracle.  Fetched
    values: per word they must be reachable -- ADD: prefix sums of a permutation; AND / OR: monotone chains between init and
    final; XOR: every fetched value is init xor (xor of a subset), checked through the multiset identity on the final."""
    npes, words, n = 4, 512, (1 << 18) + 77
    npdt, init, flat, tgt, idx, val = amo_case(width, npes, words, n, 340 + amo, distinct=False)
    mask = (1 << (8 * width)) - 1
    if amo == AMO.ADD:                                   # keep every prefix sum below 2^width so the chain check is exact
        init = (init & npdt(0xfffff)).astype(npdt)
        val = (val & np.uint64(0xf)) + np.uint64(1)
    w, ow = pair(npes, words * 8 + 4096)
    a, oa = w.malloc(words * width), ow.malloc(words * width)
    w.view(a, words * width).copy_(torch.from_numpy(init.view(np.uint8)))
    ow.view(oa, words * width, npdt)[:] = init
    f = torch.zeros(n, dtype=torch.int64, device=DEV)
    # non-fetching form first (red.global), on a copy of the state, then the fetching form (atom.global)
    w.atomic_op_batch(amo, width, a, to_dev(tgt), to_dev(idx.astype(np.int64)), val=to_dev(val.view(np.int64)))
    w.quiet(0)
    ow.amo_batch(ORC_AMO[amo], width, oa, tgt, idx, val)
    mid = ow.view(oa, words * width, npdt).copy()
    assert np.array_equal(w.view(a, words * width).cpu().numpy(), ow.view(oa, words * width))
    w.atomic_op_batch(amo, width, a, to_dev(tgt), to_dev(idx.astype(np.int64)), val=to_dev(val.view(np.int64)), fetched_out=f)
    w.quiet(0)
    ow.amo_batch(ORC_AMO[amo], width, oa, tgt, idx, val)
    fin = w.view(a, words * width).cpu().numpy().view(npdt)
    assert np.array_equal(fin, ow.view(oa, words * width, npdt))
    fet = f.cpu().numpy().view(np.uint64)
    assert (fet <= mask).all()
    v = val & np.uint64(mask)
    m0, fn = mid.reshape(-1).astype(np.uint64), fin.reshape(-1).astype(np.uint64)
    if amo == AMO.ADD:                                   # values and initial words are small here (see below): no wraparound
        from invariants import check_fetch_add
        check_fetch_add(flat, v, fet, m0, fn)
    elif amo in (AMO.AND, AMO.OR):
        # monotone: every fetched value lies between the start and the final word in the bit-lattice
        if amo == AMO.AND:
            assert ((fet & fn[flat]) == fn[flat]).all() and ((fet & m0[flat]) == fet).all()
        else:
            assert ((fet | fn[flat]) == fn[flat]).all() and ((fet | m0[flat]) == fet).all()
        # and the op that fetched the start value exists for every touched word
        first = np.zeros(npes * words, dtype=bool)
        first[flat[fet == m0[flat]]] = True
        assert first[np.unique(flat)].all()
    else:
        x = np.zeros(npes * words, dtype=np.uint64)
        np.bitwise_xor.at(x, flat, v)
        assert np.array_equal(m0 ^ x, fn)


@pytest.mark.parametrize("width", [8, 4])
@pytest.mark.parametrize("n,idx_dtype", [(1, np.int32), (1025, np.int64), (70001, np.int32)])
def test_cswap_on_distinct_words_equals_the_oracle(width, n, idx_dtype):
    """Every word is the target of at most one op, so the result does not depend on the schedule: heap and fetched values
    bit-exact against the oracle.  About half of the conditions hold; cond / val carry garbage above bit 31 (ignored on 32-bit
    words, significant on 64-bit ones)."""
    npes, words = 3, 30000
    npdt = np.uint64 if width == 8 else np.uint32
    w, ow = World(npes, words * 8 + 4096, DEV), orc.OracleWorld(npes, words * 8 + 4096)
    pad, opad = w.malloc(256), ow.malloc(256)
    a, oa = w.malloc(words * width), ow.malloc(words * width)
    init = (gen.u64(npes * words, 361) % np.uint64(2)).astype(npdt).reshape(npes, words)
    w.view(a, words * width).copy_(torch.from_numpy(init.view(np.uint8)))
    ow.view(oa, words * width, npdt)[:] = init
    flat = np.argsort(gen.u64(npes * words, 362))[:n].astype(np.int64)          # n distinct words in random order
    tgt, idx = (flat // words).astype(np.int32), (flat % words).astype(idx_dtype)
    hi = (gen.u64(n, 363) % np.uint64(2)) << np.uint64(32)
    cond = gen.u64(n, 364) % np.uint64(2) + hi
    val = gen.u64(n, 365) % np.uint64(1000) + np.uint64(2) + hi
    f = torch.zeros(n, dtype=torch.int64, device=DEV)
    w.atomic_cswap_op_batch(width, a, to_dev(tgt), to_dev(idx), f, cond=to_dev(cond.view(np.int64)), val=to_dev(val.view(np.int64)))
    w.quiet(0)
    of = ow.amo_cswap_batch(width, oa, tgt, idx, cond, val)
    assert np.array_equal(f.cpu().numpy().view(np.uint64), of)
    assert np.array_equal(w.view(a, words * width).cpu().numpy().view(npdt), ow.view(oa, words * width, npdt))
    assert 0 < int((of == (cond & np.uint64((1 << (8 * width)) - 1))).sum()) < n or n == 1


@pytest.mark.parametrize("width,empty", [(8, (1 << 64) - 1), (4, 0xffffffff)])
def test_cswap_claims_on_contended_words(width, empty):
    """Claim-style batch with scalar cond (CAS(empty -> own value)) on few words, both halves of every 64-bit cell contended
    separately on 32-bit words: exactly one winner per touched word, it fetched `empty`, the word holds its value, every loser
    fetched that value; the set of claimed words equals the oracle's."""
    from invariants import check_compare_swap_claim
    npes, words, n = 2, 500, 300001
    npdt = np.uint64 if width == 8 else np.uint32
    w, ow = World(npes, words * 8 + 4096, DEV), orc.OracleWorld(npes, words * 8 + 4096)
    a, oa = w.malloc(words * width), ow.malloc(words * width)
    w.view(a, words * width).fill_(255)
    ow.view(oa, words * width, npdt)[:] = empty
    flat = (gen.u64(n, 366) % np.uint64(npes * words - 7)).astype(np.int64)     # the last 7 words stay untouched
    tgt, idx = (flat // words).astype(np.int32), (flat % words).astype(np.int32)
    val = (np.arange(n, dtype=np.uint64) + np.uint64(1)) & np.uint64(0x7fffffff)
    f = torch.zeros(n, dtype=torch.int64, device=DEV)
    w.atomic_cswap_op_batch(width, a, to_dev(tgt), to_dev(idx), f, cond_scalar=empty, val=to_dev(val.view(np.int64)))
    w.quiet(0)
    fin = w.view(a, words * width).cpu().numpy().view(npdt).reshape(-1).astype(np.uint64)
    check_compare_swap_claim(flat, val, f.cpu().numpy().view(np.uint64), fin, empty=empty)
    ow.amo_cswap_batch(width, oa, tgt, idx, np.full(n, empty, dtype=np.uint64), val)
    ofin = ow.view(oa, words * width, npdt).reshape(-1).astype(np.uint64)
    assert np.array_equal(fin == np.uint64(empty), ofin == np.uint64(empty))
    with pytest.raises(ShmemgError):
        w.atomic_cswap_op_batch(2, a, to_dev(tgt), to_dev(idx), f)                # no 16-bit words
    with pytest.raises(ShmemgError):
        w.atomic_cswap_op_batch(4, a + 2, to_dev(tgt), to_dev(idx), f)            # misaligned
    w.atomic_cswap_op_batch(4, a, to_dev(tgt[:0]), to_dev(idx[:0]), f[:0])        # no ops: nothing enqueued


@pytest.mark.parametrize("idx_dtype", [np.int32, np.int64])
def test_amo_check_batch_finds_the_first_out_of_range_op(idx_dtype):
    """The device-side bounds check of the SoA index arrays (the host cannot see them): None when every op is in bounds, else
    the smallest offending op index; the last whole word of the window is in bounds, the one after it is not."""
    npes, hb, n = 3, 4096 + 24, 50001                       # 515 whole 64-bit words, 1030 32-bit words per window
    w = World(npes, hb, DEV)
    off = 256
    tgt = gen.uniform_i32(n, 0, npes - 1, 371, 0)
    for width, last in ((8, (hb - off) // 8 - 1), (4, (hb - off) // 4 - 1)):
        idx = (gen.u64(n, 372) % np.uint64(last + 1)).astype(idx_dtype)
        idx[123] = last                                      # the last whole word: fine
        assert w.amo_check_batch(width, off, to_dev(tgt), to_dev(idx)) is None
        bad = idx.copy(); bad[40000] = last + 1; bad[777] = last + 1
        assert w.amo_check_batch(width, off, to_dev(tgt), to_dev(bad)) == 777
        t2 = tgt.copy(); t2[31] = npes; t2[9000] = -1
        assert w.amo_check_batch(width, off, to_dev(t2), to_dev(bad)) == 31
        neg = idx.copy(); neg[n - 1] = -1                    # a negative index is a huge unsigned one
        assert w.amo_check_batch(width, off, to_dev(tgt), to_dev(neg)) == n - 1
    assert w.amo_check_batch(8, off, to_dev(tgt[:0]), to_dev(idx[:0])) is None
    with pytest.raises(ShmemgError):
        w.amo_check_batch(8, off + 4, to_dev(tgt), to_dev(idx))


@pytest.mark.parametrize("width", [8, 4])
def test_generic_amo_swap_chain_set_and_fetch(width):
    npes, words, n = 3, 64, 50000
    npdt = np.uint64 if width == 8 else np.uint32
    w = World(npes, words * 8 + 4096, DEV)
    a = w.malloc(words * width)
    init = (np.arange(npes * words, dtype=np.uint64) + np.uint64(1 << 30)).astype(npdt).reshape(npes, words)
    w.view(a, words * width).copy_(torch.from_numpy(init.view(np.uint8)))
    flat = (gen.u64(n, 351) % np.uint64(npes * words)).astype(np.int64)
    tgt, idx = to_dev((flat // words).astype(np.int32)), to_dev((flat % words).astype(np.int32))
    val = np.arange(1, n + 1, dtype=np.uint64)
    f = torch.zeros(n, dtype=torch.int64, device=DEV)
    w.atomic_op_batch(AMO.SWAP, width, a, tgt, idx, val=to_dev(val.view(np.int64)), fetched_out=f)
    w.quiet(0)
    fin = w.view(a, words * width).cpu().numpy().view(npdt).reshape(-1).astype(np.uint64)
    fet = f.cpu().numpy().view(np.uint64)
    # per word: {fetched} + {final} == {init} + {swapped-in values}  (a chain of exchanges permutes the values)
    got = np.sort(np.concatenate([flat * (1 << 32) + fet.astype(np.int64), np.arange(npes * words) * (1 << 32) + fin.astype(np.int64)]))
    exp = np.sort(np.concatenate([flat * (1 << 32) + val.astype(np.int64),
                                  np.arange(npes * words) * (1 << 32) + init.reshape(-1).astype(np.int64)]))
    assert np.array_equal(got, exp)
    # atomic_fetch: values equal the words, which stay unchanged; scalar value + no fetch = atomic_set / atomic_inc
    g = torch.zeros(n, dtype=torch.int64, device=DEV)
    w.atomic_op_batch(AMO.FETCH, width, a, tgt, idx, fetched_out=g)
    w.quiet(0)
    assert np.array_equal(g.cpu().numpy().view(np.uint64), fin[flat])
    assert np.array_equal(w.view(a, words * width).cpu().numpy().view(npdt).reshape(-1).astype(np.uint64), fin)
    w.atomic_op_batch(AMO.ADD, width, a, tgt, idx, val_scalar=1)                  # atomic_inc
    w.quiet(0)
    cnt = np.bincount(flat, minlength=npes * words).astype(np.uint64)
    assert np.array_equal(w.view(a, words * width).cpu().numpy().view(npdt).reshape(-1).astype(np.uint64),
                          (fin + cnt) & np.uint64((1 << (8 * width)) - 1))
    w.atomic_op_batch(AMO.SWAP, width, a, tgt, idx, val_scalar=77)                # atomic_set
    w.quiet(0)
    out = w.view(a, words * width).cpu().numpy().view(npdt).reshape(-1)
    assert (out[np.unique(flat)] == 77).all()
    with pytest.raises(ShmemgError):
        w.atomic_op_batch(AMO.FETCH, width, a, tgt, idx)                          # FETCH needs an output array
    with pytest.raises(ShmemgError):
        w.atomic_op_batch(AMO.ADD, 8, a + 4, tgt, idx, val_scalar=1)              # misaligned 64-bit words


# ---- block-strided put / get -----------------------------------------------------------------------------------------
@pytest.mark.parametrize("block,ds,ss,nb,do,so", [
    (8, 8, 2048, 65536, 0, 0),            # element path: the z-face gather of a 256^3 cube (stride 2 KiB -> contiguous)
    (8, 2048, 8, 4097, 8, 16),            # element path: scatter
    (4, 12, 20, 10001, 4, 8), (16, 48, 16, 7777, 16, 32),
    (2048, 2048, 524288, 256, 0, 0),      # bulk path: the y-face of a 256^3 cube (256 rows of 2 KiB)
    (65536 + 32, 65536 + 64, 131072, 9, 16, 48),   # bulk path, blocks longer than one tile
    (1000, 1000, 1024, 300, 3, 5),        # generic path: odd sizes and alignments
    (3, 7, 5, 5000, 1, 2), (1, 1, 3, 100, 0, 1), (24, 24, 40, 999, 8, 8),
    (8, 8, 8, 0, 0, 0), (0, 8, 8, 10, 0, 0),
])
@pytest.mark.parametrize("get", [False, True])
def test_ibput_ibget_match_oracle(block, ds, ss, nb, do, so, get):
    npes = 3
    dspan = (max(nb - 1, 0) * ds + block + do + 64 + 255) // 256 * 256
    sspan = (max(nb - 1, 0) * ss + block + so + 64 + 255) // 256 * 256
    w, ow = pair(npes, dspan + sspan + 4096)
    s, d = w.malloc(sspan), w.malloc(dspan)
    os_, od = ow.malloc(sspan), ow.malloc(dspan)
    fill(w, ow, s, os_, sspan, 360)
    w.view(d, dspan).zero_()
    if get:
        w.ibget(d + do, s + so, ds, ss, block, nb, 1, 2)
        ow.ibget(od + do, os_ + so, ds, ss, block, nb, 1, 2)
    else:
        w.ibput(d + do, s + so, ds, ss, block, nb, 0, 2)
        ow.ibput(od + do, os_ + so, ds, ss, block, nb, 0, 2)
    w.quiet(0)
    assert np.array_equal(w.view(d, dspan).cpu().numpy(), ow.view(od, dspan))
    assert np.array_equal(w.view(s, sspan).cpu().numpy(), ow.view(os_, sspan))


def test_ibput_moves_the_three_halo_faces_without_a_pack_kernel():
    """C2's faces straight out of the cube (B = 64): x-face = one block, y-face = B blocks of B elements, z-face = B^2 single
    elements at stride B; each equals the numpy slice of the cube."""
    B = 64
    w = World(2, B ** 3 * 8 + 3 * B * B * 8 + 4096, DEV)
    U, fx, fy, fz = w.malloc(B ** 3 * 8), w.malloc(B * B * 8), w.malloc(B * B * 8), w.malloc(B * B * 8)
    cube = gen.u64(2 * B ** 3, 361).reshape(2, B, B, B)
    w.view(U, B ** 3 * 8, torch.int64).copy_(torch.from_numpy(cube.reshape(2, -1).view(np.int64)))
    w.ibput(fx, U + (B - 1) * B * B * 8, 0, 0, B * B * 8, 1, 0, 1)
    w.ibput(fy, U + 5 * B * 8, B * 8, B * B * 8, B * 8, B, 0, 1)
    w.ibput(fz, U + (B - 1) * 8, 8, B * 8, 8, B * B, 0, 1)
    w.quiet(0)
    got = lambda off: w.view(off, B * B * 8, torch.int64).cpu().numpy().view(np.uint64)[1].reshape(B, B)   # noqa: E731
    assert np.array_equal(got(fx), cube[0, B - 1]) and np.array_equal(got(fy), cube[0, :, 5, :])
    assert np.array_equal(got(fz), cube[0, :, :, B - 1])
    with pytest.raises(ShmemgError):
        w.ibput(fz, U, 8, B * 8, 8, B * B * B, 0, 1)          # runs out of the window
    with pytest.raises(ShmemgError):
        w.ibput(fz, U, 8, 8, 8, 4, 0, 2)                      # PE out of range


# ---- signal test -------------------------------------------------------------------------------------------------------
def test_signal_test_truth_table_and_acquire():
    w = World(2, 1 << 16, DEV)
    ow = orc.OracleWorld(2, 1 << 16)
    data, sig = w.malloc(4096), w.calloc(2, 8)
    odata, osig = ow.malloc(4096), ow.malloc(16)
    res = torch.full((1,), -1, dtype=torch.int32, device=DEV)
    w.signal_test(sig + 8, CMP.EQ, 0, 1, res)
    w.quiet(0)
    assert res.item() == 1 and ow.signal_test(osig + 8, CMP.EQ, 0, 1)
    w.put_signal(data, data, 4096, sig + 8, 5, SIGNAL.SET, 0, 1)
    ow.view(osig, 16, np.uint64)[1, 1] = 5
    for cmp in (CMP.EQ, CMP.NE, CMP.GT, CMP.GE, CMP.LT, CMP.LE):
        for v in (4, 5, 6, M64):
            w.signal_test(sig + 8, cmp, v, 1, res)
            w.quiet(0)
            assert res.item() == int(ow.signal_test(osig + 8, cmp, v, 1)), (cmp, v)
    with pytest.raises(ShmemgError):
        w.signal_test(sig + 4, CMP.EQ, 0, 1, res)
    with pytest.raises(ShmemgError):
        w.signal_test(sig, 9, 0, 1, res)


def test_reduce_signed_zero_corner_matches_oracle():
    npes = 3
    w, ow = pair(npes, 4096)
    s, d = w.malloc(256), w.malloc(256)
    os_, od = ow.malloc(256), ow.malloc(256)
    x = np.full((npes, 8), -0.0, dtype=np.float32)
    x[1, 4:] = 0.0
    w.view(s, 32, torch.float32).copy_(torch.from_numpy(x))
    ow.view(os_, 32, np.float32)[:] = x
    for op in (RED.SUM, RED.PROD, RED.MIN, RED.MAX):
        w.reduce(op, F32, d, s, 8)
        w.quiet(0)
        ow.reduce(ORC_OP[op], "f32", od, os_, 8)
        g, o = w.view(d, 32).cpu().numpy().view(np.uint32), ow.view(od, 32, np.uint32)
        if op in (RED.MIN, RED.MAX):                     # min(-0, +0): either zero is a correct result
            assert np.array_equal(g[:, :4], o[:, :4]) and (g[:, 4:] & 0x7fffffff == 0).all()
        else:
            assert np.array_equal(g, o), op


# ---- vector test / wait ------------------------------------------------------------------------------------------------
def test_vector_test_and_wait_forms_match_oracle():
    npes, n = 3, 700
    w, ow = pair(npes, 1 << 16)
    sig, osig = w.calloc(n, 8), ow.malloc(n * 8)
    vals = (gen.u64(npes * n, 371) % np.uint64(5)).reshape(npes, n)
    w.view(sig, n * 8, torch.int64).copy_(torch.from_numpy(vals.view(np.int64)))
    ow.view(osig, n * 8, np.uint64)[:] = vals
    idx = torch.full((n,), -1, dtype=torch.int64, device=DEV)
    cnt = torch.full((1,), -1, dtype=torch.int64, device=DEV)
    for cmp in (CMP.EQ, CMP.NE, CMP.GT, CMP.GE, CMP.LT, CMP.LE):
        for v, pe, off, m in ((2, 0, 0, n), (0, 1, 8 * 3, n - 7), (4, 2, 8 * 100, 257), (9, 1, 0, 1), (1, 0, 8, 0)):
            w.signal_test_vec(sig + off, m, cmp, v, pe, idx, cnt)
            w.quiet(0)
            exp = ow.signal_test_vec(osig + off, m, cmp, v, pe)
            assert cnt.item() == len(exp) and np.array_equal(idx.cpu().numpy()[:len(exp)].view(np.uint64), exp), (cmp, v, pe)
    # wait_until_all on words that a put_signal chain sets one by one (stream order makes them all true before the wait)
    data = w.malloc(4096)
    w.view(sig, n * 8).zero_()
    for k in range(6):
        w.put_signal(data, data, 64, sig + 8 * k, k + 1, SIGNAL.SET, 0, 2)
    w.signal_wait_until_all(sig, 6, CMP.GE, 1, 2)
    w.signal_wait_until_some(sig, 10, CMP.GE, 4, 2, idx, cnt)
    w.quiet(0)
    ow.view(osig, n * 8, np.uint64)[:] = 0
    ow.view(osig, n * 8, np.uint64)[2, :6] = np.arange(1, 7)
    exp = ow.signal_test_vec(osig, 10, CMP.GE, 4, 2)
    assert cnt.item() == 3 and np.array_equal(idx.cpu().numpy()[:3].view(np.uint64), exp) and exp.tolist() == [3, 4, 5]
    with pytest.raises(ShmemgError):
        w.signal_test_vec(sig + 4, 2, CMP.EQ, 0, 0)
    with pytest.raises(ShmemgError):
        w.signal_wait_until_all(sig, 1 << 40, CMP.EQ, 0, 0)
