"""Pins of the CPU oracle against things other than itself (CPU only; no GPU, no CUDA package).

The paper prints no numeric example, so each part is pinned by what the mathematics
fixes: library routines (numpy slice assignment, np.add.at, np.sum, math.fsum, np.concatenate),
closed forms (transpose identity, involution, N*c), hand-computed 2-PE programs with the expected heaps
written out, and schedule-independent invariants.  SURVEY.md 8(c) "What pins each part".
"""
import math

import numpy as np
import pytest

from invariants import check_compare_swap_claim, check_fetch_add
from oracle import oracle as orc
from workloads import configs, gen
from workloads.spec import CMP_EQ, CMP_GE, CMP_GT, CMP_LE, CMP_LT, CMP_NE, SIGNAL_ADD, SIGNAL_SET, Program

M64 = (1 << 64) - 1


def run(prog, heap_bytes=None):
    hb = heap_bytes or (sum((b + 255) // 256 * 256 for b in prog.obj_bytes) + 256)
    w = orc.OracleWorld(prog.npes, hb)
    w.load_program(prog)
    w.run_program(prog)
    return w


# ---- hand-computed programs (expected heaps written out) -------------------------------------------
def test_hand_put_get_two_pes():
    p = Program(2)
    p.obj("a", 32, np.array([[1, 2, 3, 4], [10, 20, 30, 40]], dtype=np.uint64))
    p.put(0, 1, ("a", 0), ("a", 8), 16)      # PE1.a[0:2] = PE0.a[1:3] = 2,3
    p.get(0, 1, ("a", 24), ("a", 0), 8)      # PE0.a[3] = PE1.a[0] = 2
    p.put(1, 0, ("a", 0), ("a", 24), 8)      # PE0.a[0] = PE1.a[3] = 40
    w = run(p)
    assert w.obj("a", np.uint64).tolist() == [[40, 2, 3, 2], [2, 3, 30, 40]]


def test_hand_amo_and_signal():
    p = Program(2)
    p.obj("x", 32, np.array([[5, 0, 0, 0], [7, M64, 0, 0]], dtype=np.uint64))
    p.atomic_add(0, 1, ("x", 0), 3)                       # PE1.x0 = 10
    p.atomic_fetch_add(1, 1, ("x", 0), M64, ("x", 16))    # adds -1: PE1.x0 = 9, PE1.x2 = 10
    p.atomic_compare_swap(0, 1, ("x", 8), M64, 77, ("x", 8))   # PE1.x1: -1 -> 77, PE0.x1 = -1
    p.atomic_compare_swap(1, 1, ("x", 8), M64, 88, ("x", 24))  # fails, PE1.x3 = 77
    p.put_signal(0, 1, ("x", 16), ("x", 0), 8, ("x", 24), 5, SIGNAL_ADD)   # PE1.x2 = 5, PE1.x3 = 82
    p.put_signal(0, 1, ("x", 16), ("x", 0), 8, ("x", 0), 1, SIGNAL_SET)    # PE1.x0 = 1
    w = run(p)
    assert w.obj("x", np.uint64).tolist() == [[5, M64, 0, 0], [1, 77, 5, 82]]


def test_hand_wraparound_add():
    p = Program(2)
    p.obj("x", 8, np.array([[M64], [M64 - 1]], dtype=np.uint64))
    p.atomic_add(0, 0, ("x", 0), 2)
    p.atomic_add(0, 1, ("x", 0), 5)
    w = run(p)
    assert w.obj("x", np.uint64).ravel().tolist() == [1, 3]


@pytest.mark.parametrize("cmp,val,ok", [(CMP_EQ, 5, True), (CMP_EQ, 4, False), (CMP_NE, 4, True), (CMP_NE, 5, False),
                                        (CMP_GT, 4, True), (CMP_GT, 5, False), (CMP_GE, 5, True), (CMP_GE, 6, False),
                                        (CMP_LT, 6, True), (CMP_LT, 5, False), (CMP_LE, 5, True), (CMP_LE, 4, False),
                                        (CMP_GT, M64, False), (CMP_LT, M64, True)])   # unsigned compare
def test_wait_until_comparisons(cmp, val, ok):
    p = Program(1)
    p.obj("s", 8, np.array([[5]], dtype=np.uint64))
    p.signal_wait_until(0, ("s", 0), cmp, val)
    if ok:
        run(p)
    else:
        with pytest.raises(orc.OracleError, match="WAIT_UNSATISFIED at op 0"):
            run(p)


def test_range_and_alignment_errors():
    p = Program(2)
    p.obj("a", 64)
    p.put(0, 1, ("a", 32), ("a", 0), 64)        # runs off the end of a 256-byte heap
    with pytest.raises(orc.OracleError, match="RANGE"):
        run(p, heap_bytes=64)
    q = Program(2)
    q.obj("a", 64)
    q.atomic_add(0, 1, ("a", 4), 1)
    with pytest.raises(orc.OracleError, match="ALIGN"):
        run(q)
    r = Program(2)
    r.obj("a", 64)
    r.put(0, 2, ("a", 0), ("a", 0), 8)
    with pytest.raises(orc.OracleError, match="RANGE"):
        run(r)


# ---- put/get against numpy slice assignment, random offsets and sizes ------------------------------------
def test_put_get_random_vs_numpy():
    npes, nb, nops = 5, 4096, 300
    rng = np.random.default_rng(7)
    init = rng.integers(0, 256, size=(npes, nb), dtype=np.uint8)
    p = Program(npes)
    p.obj("m", nb, init)
    ref = init.copy()
    for _ in range(nops):
        i, t = rng.integers(0, npes, 2)
        n = int(rng.integers(0, 300))
        d, s = int(rng.integers(0, nb - n + 1)), int(rng.integers(0, nb - n + 1))
        if rng.integers(0, 2):
            p.put(int(i), int(t), ("m", d), ("m", s), n)
            ref[t, d:d + n] = ref[i, s:s + n].copy()
        else:
            p.get(int(i), int(t), ("m", d), ("m", s), n)
            ref[i, d:d + n] = ref[t, s:s + n].copy()
    w = run(p)
    assert np.array_equal(w.obj("m"), ref)


# ---- collectives: closed forms ------------------------------------------------------------------------------
@pytest.mark.parametrize("npes,blk", [(2, 8), (5, 24), (16, 1000), (64, 96)])
def test_alltoall_transpose_identity_and_involution(npes, blk):
    w = orc.OracleWorld(npes, 3 * npes * blk + 1024)
    a = w.malloc(npes * blk)
    b = w.malloc(npes * blk)
    c = w.malloc(npes * blk)
    src = gen.u64((npes * npes * blk + 7) // 8, 21).view(np.uint8)[:npes * npes * blk].reshape(npes, npes * blk)
    w.view(a, npes * blk)[:] = src
    w.alltoall(b, a, blk)
    exp = src.reshape(npes, npes, blk).transpose(1, 0, 2).reshape(npes, npes * blk)
    assert np.array_equal(w.view(b, npes * blk), exp)
    assert np.array_equal(w.view(a, npes * blk), src)          # source untouched
    w.alltoall(c, b, blk)
    assert np.array_equal(w.view(c, npes * blk), src)          # alltoall(alltoall(x)) = x


def test_alltoall_equals_put_program():
    npes, blk = 6, 40
    payload = configs.c3a_payload(npes, blk, seed=2)
    prog = configs.c3a_put_program(npes, blk, payload=payload)
    w = run(prog)
    exp = payload.reshape(npes, npes, blk).transpose(1, 0, 2).reshape(npes, npes * blk)
    assert np.array_equal(w.obj("dst"), exp)


def test_alltoall_rejects_overlap():
    w = orc.OracleWorld(4, 4096)
    with pytest.raises(orc.OracleError):
        w.alltoall(64, 0, 32)       # 4*32 = 128 bytes from 0 overlaps dst at 64


@pytest.mark.parametrize("npes,n", [(1, 16), (3, 5), (128, 64)])
def test_fcollect_is_concatenation(npes, n):
    w = orc.OracleWorld(npes, npes * n + n + 1024)
    s = w.malloc(n)
    d = w.malloc(npes * n)
    src = np.random.default_rng(3).integers(0, 256, size=(npes, n), dtype=np.uint8)
    w.view(s, n)[:] = src
    w.fcollect(d, s, n)
    cat = np.concatenate([src[p] for p in range(npes)])
    for j in range(npes):
        assert np.array_equal(w.view(d, npes * n)[j], cat)


def test_sum_reduce_i64_vs_numpy_and_constant():
    npes, n = 17, 1000
    w = orc.OracleWorld(npes, 2 * 8 * n + 1024)
    s, d = w.malloc(8 * n), w.malloc(8 * n)
    x = configs.c5_i64(npes, n)
    w.view(s, 8 * n, np.int64)[:] = x
    w.sum_reduce_i64(d, s, n)
    exp = np.sum(x, axis=0, dtype=np.int64)
    for j in range(npes):
        assert np.array_equal(w.view(d, 8 * n, np.int64)[j], exp)
    w.view(s, 8 * n, np.int64)[:] = -12345
    w.sum_reduce_i64(d, s, n)
    assert (w.view(d, 8 * n, np.int64) == -12345 * npes).all()
    # wraparound: 4 * 2^62 = 2^64 = 0
    w.view(s, 8 * n, np.int64)[:] = 0
    w.view(s, 8 * n, np.int64)[:4] = 1 << 62
    w.sum_reduce_i64(d, s, n)
    assert (w.view(d, 8 * n, np.int64) == 0).all()
    # in-place (exact aliasing is allowed for sum_reduce, reading 12)
    w.view(s, 8 * n, np.int64)[:] = x
    w.sum_reduce_i64(s, s, n)
    assert np.array_equal(w.view(s, 8 * n, np.int64)[3], exp)


def test_sum_reduce_f32_vs_fsum():
    npes, n = 128, 4096
    w = orc.OracleWorld(npes, 2 * 4 * n + 1024)
    s, d = w.malloc(4 * n), w.malloc(4 * n)
    x = configs.c5_f32(npes, n)
    w.view(s, 4 * n, np.float32)[:] = x
    r64 = w.sum_reduce_f32(d, s, n, want_r64=True)
    out = w.view(d, 4 * n, np.float32)
    assert (out == out[0]).all()                                   # all PEs hold identical results
    for k in range(0, n, 7):
        exact = math.fsum(float(v) for v in x[:, k])               # exactly rounded fp64 sum
        # 128 fp64 adds of |x| < 8: error far below fp32 resolution; relative bound from the arithmetic:
        assert abs(r64[k] - exact) <= 128 * 2.0 ** -53 * float(np.abs(x[:, k]).astype(np.float64).sum())
        assert out[0, k] == np.float32(r64[k])
    # exactly representable case: small integers sum exactly
    xi = (gen.uniform_i64(npes * n, -1000, 1000, 5).reshape(npes, n)).astype(np.float32)
    w.view(s, 4 * n, np.float32)[:] = xi
    w.sum_reduce_f32(d, s, n)
    assert np.array_equal(w.view(d, 4 * n, np.float32)[5], xi.astype(np.int64).sum(axis=0).astype(np.float32))


# ---- atomics ----------------------------------------------------------------------------------------------------
def test_c1_atomic_add_vs_numpy_add_at():
    wl = configs.c1_atomic_add()            # the full config-1 workload: 65 536 ops, 4 PEs x 16 384 int64
    w = orc.OracleWorld(wl.npes, wl.nelem * 8 + 256)
    a = w.malloc(wl.nelem * 8)
    w.atomic_add_batch(a, wl.tgt_pe, wl.idx, wl.val)
    exp = np.zeros((wl.npes, wl.nelem), dtype=np.int64)
    np.add.at(exp, (wl.tgt_pe, wl.idx.astype(np.int64)), wl.val)
    assert np.array_equal(w.view(a, wl.nelem * 8, np.int64), exp)
    assert int(exp.sum()) == int(wl.val.sum())
    # same thing through the general descriptor path
    p = Program(wl.npes)
    p.obj("A", wl.nelem * 8)
    for i in range(4096):
        p.atomic_add(i % wl.npes, int(wl.tgt_pe[i]), ("A", int(wl.idx[i]) * 8), int(wl.val[i]))
    w2 = run(p)
    exp2 = np.zeros((wl.npes, wl.nelem), dtype=np.int64)
    np.add.at(exp2, (wl.tgt_pe[:4096], wl.idx[:4096].astype(np.int64)), wl.val[:4096])
    assert np.array_equal(w2.obj("A", np.int64), exp2)


def test_fetch_add_and_cas_on_small_graph():
    g = configs.c4_graph(scale=10, edge_factor=16, npes=8)
    vpp = g.verts_per_pe
    w = orc.OracleWorld(g.npes, 2 * vpp * 8 + 512)
    deg, par = w.malloc(vpp * 8), w.malloc(vpp * 8)
    w.view(par, vpp * 8, np.uint64)[:] = M64
    E = len(g.u)
    ones = np.ones(E, dtype=np.uint64)
    f_deg = w.atomic_fetch_add_batch(deg, g.owner(g.u), g.local(g.u), ones)
    f_par = w.atomic_compare_swap_batch(par, g.owner(g.v), g.local(g.v), np.full(E, M64, dtype=np.uint64),
                                        g.u.astype(np.uint64))
    degs = w.view(deg, vpp * 8, np.uint64).reshape(-1)
    pars = w.view(par, vpp * 8, np.uint64).reshape(-1)
    # library pins
    assert np.array_equal(degs, np.bincount(g.u, minlength=1 << g.scale).astype(np.uint64))
    # sequential schedule: fetched degree = number of earlier occurrences of u
    order = np.argsort(g.u, kind="stable")
    us = g.u[order]
    start = np.r_[0, np.flatnonzero(us[1:] != us[:-1]) + 1]
    rank = np.arange(E) - np.repeat(start, np.diff(np.r_[start, E]))
    exp_f = np.empty(E, dtype=np.uint64)
    exp_f[order] = rank.astype(np.uint64)
    assert np.array_equal(f_deg, exp_f)
    # CAS: oracle's winner = first occurrence in batch order
    uniq, first = np.unique(g.v, return_index=True)
    exp_par = np.full(1 << g.scale, M64, dtype=np.uint64)
    exp_par[uniq] = g.u[first]
    assert np.array_equal(pars, exp_par)
    # schedule-independent invariants hold for the oracle's schedule too
    check_fetch_add(g.u.astype(np.int64), ones, f_deg, np.zeros(1 << g.scale, dtype=np.uint64), degs)
    check_compare_swap_claim(g.v.astype(np.int64), g.u.astype(np.uint64), f_par, pars)
    # every claimed parent is a valid in-neighbour
    claimed = np.flatnonzero(pars != M64)
    edges = set(zip(g.u.tolist(), g.v.tolist()))
    assert all((int(pars[v]), int(v)) in edges for v in claimed[:2000])


def test_invariant_checkers_reject_wrong_outputs():
    key = np.array([0, 0, 0, 1])
    val = np.array([2, 3, 4, 1], dtype=np.uint64)
    init = np.array([10, 0], dtype=np.uint64)
    good = np.array([13, 10, 15, 0], dtype=np.uint64)          # order: op1 (10), op0 (13), op2 (15)
    check_fetch_add(key, val, good, init, np.array([19, 1], dtype=np.uint64))
    with pytest.raises(AssertionError):
        check_fetch_add(key, val, np.array([12, 10, 15, 0], dtype=np.uint64), init, np.array([19, 1], dtype=np.uint64))
    with pytest.raises(AssertionError):
        check_fetch_add(key, val, good, init, np.array([18, 1], dtype=np.uint64))
    with pytest.raises(AssertionError):                         # duplicate fetched value = lost update
        check_fetch_add(key, val, np.array([10, 10, 15, 0], dtype=np.uint64), init, np.array([19, 1], dtype=np.uint64))
    ck = np.array([0, 0, 2])
    cv = np.array([5, 6, 7], dtype=np.uint64)
    fin = np.array([6, M64, 7], dtype=np.uint64)
    check_compare_swap_claim(ck, cv, np.array([6, M64, M64], dtype=np.uint64), fin)
    with pytest.raises(AssertionError):                         # two winners
        check_compare_swap_claim(ck, cv, np.array([M64, M64, M64], dtype=np.uint64), fin)
    with pytest.raises(AssertionError):                         # final is the loser's value
        check_compare_swap_claim(ck, cv, np.array([6, M64, M64], dtype=np.uint64), np.array([5, M64, 7], dtype=np.uint64))
    with pytest.raises(AssertionError):                         # untouched slot modified
        check_compare_swap_claim(ck, cv, np.array([6, M64, M64], dtype=np.uint64), np.array([6, 1, 7], dtype=np.uint64))


# ---- halo application compute --------------------------------------------------------------------------------------
def test_halo_pack_perturb_checksum():
    B = 6
    h = configs.Halo(B)
    U0 = h.initial_U()
    for p in (0, 3, 7):
        U = U0[p].copy()
        orc.halo_perturb(U, B, h.coord(p), h.seed, 4)
        px, py, pz = h.coord(p)
        G = 2 * B
        x, y, z = np.meshgrid(np.arange(B), np.arange(B), np.arange(B), indexing="ij")
        g = ((px * B + x) * G + (py * B + y)) * G + (pz * B + z)
        # the generator module's mix64 is an independent implementation of the same counter-based hash
        delta = np.array([(gen.mix64(h.seed, 4, int(i)) & 0xFFFF) * 2.0 ** -30 for i in g.ravel()])
        assert np.array_equal(U, U0[p] + delta)
        assert 0 <= delta.min() and delta.max() < 2.0 ** -14
        cube = U.reshape(B, B, B)
        faces = [cube[0, :, :], cube[B - 1, :, :], cube[:, 0, :], cube[:, B - 1, :], cube[:, :, 0], cube[:, :, B - 1]]
        for f in range(6):
            send = np.empty(B * B)
            orc.halo_pack(U, B, f, send)
            assert np.array_equal(send, faces[f].reshape(-1))
    a = gen.u64(37, 9)
    assert orc.checksum64(a) == sum(int(v) * (2 * k + 1) for k, v in enumerate(a)) & M64


def test_halo_round_program_delivers_neighbour_faces():
    B = 4
    h = configs.Halo(B)
    prog = h.program(with_consume=True, with_U=False)
    fb = h.face_bytes
    w = orc.OracleWorld(8, 64 * fb)
    w.load_program(prog)
    send = w.obj("send", np.float64)
    for rnd in (1, 2, 3):
        send[:] = gen.uniform_f64(8 * 6 * B * B, 50 + rnd).reshape(8, -1)
        w.run_program(h.round_ops(prog, rnd, with_consume=True))
        ghost = w.obj("ghost", np.float64).reshape(8, 2, 6, B * B)
        cons = w.obj("consumed", np.float64).reshape(8, 6, B * B)
        s = send.reshape(8, 6, B * B)
        for p in range(8):
            for axis in range(3):
                q = p ^ (4 >> axis)
                # my low-side ghost (slot 2*axis+0) holds the neighbour's HIGH face (2*axis+1) and vice versa
                assert np.array_equal(ghost[p, rnd & 1, 2 * axis + 0], s[q, 2 * axis + 1])
                assert np.array_equal(ghost[p, rnd & 1, 2 * axis + 1], s[q, 2 * axis + 0])
        assert np.array_equal(cons, ghost[:, rnd & 1])
        assert (w.obj("sig", np.uint64) == rnd).all()


# ---- generators: determinism and the distributions the configs name ------------------------------------------------
def test_generators():
    assert np.array_equal(gen.u64(1000, 5, 2), gen.u64(1000, 5, 2))
    assert np.array_equal(gen.u64(1000, 5, 2)[100:], gen.u64(900, 5, 2, i0=100))     # counter-based
    assert not np.array_equal(gen.u64(1000, 5, 2), gen.u64(1000, 5, 3))
    v = gen.uniform_i64(200000, 1, 1000, 0, 2)
    assert v.min() == 1 and v.max() == 1000 and abs(v.mean() - 500.5) < 3
    f = gen.uniform_f64(200000, 1)
    assert 0 <= f.min() and f.max() < 1 and abs(f.mean() - 0.5) < 0.005
    n = gen.normal_f32(400000, 4).astype(np.float64)
    assert abs(n.mean()) < 0.01 and abs(n.std() - 1) < 0.01
    b = gen.normal_bf16_bits(100000, 2)
    bf = (b.astype(np.uint32) << 16).view(np.float32).astype(np.float64)
    assert abs(bf.mean()) < 0.02 and abs(bf.std() - 1) < 0.02
    u, vv = gen.rmat_edges(1 << 16, 12)
    assert u.max() < (1 << 12) and vv.max() < (1 << 12)
    top_u = (u >> 11) & 1
    assert abs(top_u.mean() - 0.24) < 0.01            # P(u bit = 1) = c + d = 0.24  (Appendix D)
    assert abs(((vv >> 11) & 1).mean() - 0.24) < 0.01
    k = gen.zipf_ranks(200000, 1.1, 64, 2, 1)
    wts = np.arange(1, 65) ** -1.1
    assert k.min() == 1 and k.max() == 64 and abs(k.mean() - (wts * np.arange(1, 65)).sum() / wts.sum()) < 0.2
    sk = configs.c3b_skewed(npes=8)
    assert (sk.sizes % 4096 == 0).all() and sk.sizes.min() >= 4096 and sk.sizes.max() <= 262144
