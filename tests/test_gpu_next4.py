"""GPU parity of SURVEY.md 8(f) NEXT-4: the block-strided alltoall (FFT-style transposes) and the CPU space of the
two-space model, against the CPU oracle; the oracle routines are pinned in tests/test_oracle_pins_next4.py."""
import numpy as np
import pytest
import torch

from gpu_common import DEV
from oracle import oracle as orc
from paper_2607_08006_b200 import CAP, ERR, TEAM, ShmemgError, World
from workloads import configs, gen

pytestmark = pytest.mark.gpu


def _pair(npes, hb):
    return World(npes, hb, DEV), orc.OracleWorld(npes, hb)


@pytest.mark.parametrize("npes,X,Y,Z,es", [(4, 8, 12, 5, 8), (8, 64, 64, 64, 8), (16, 32, 48, 200, 8), (3, 6, 9, 7, 4), (64, 128, 128, 32, 8)])
def test_fft_transpose_matches_oracle_and_numpy(npes, X, Y, Z, es):
    t = configs.fft_transpose(npes, X, Y, Z, es, seed=11)
    sb = t.slab_bytes
    w, ow = _pair(npes, 2 * sb + 8192)
    s, d = w.malloc(sb), w.malloc(sb)
    os_, od = ow.malloc(sb), ow.malloc(sb)
    w.view(s, sb).copy_(torch.from_numpy(t.A)); ow.view(os_, sb)[:] = t.A
    w.view(d, sb).zero_()
    block, nblocks, sbs, sps, dbs, dps = t.params()
    w.alltoalls(d, s, dps, sps, dbs, sbs, block, nblocks)
    ow.alltoalls(od, os_, dps, sps, dbs, sbs, block, nblocks)
    w.quiet(0)
    got = w.view(d, sb).cpu().numpy()
    assert np.array_equal(got, ow.view(od, sb))
    ut = {4: np.uint32, 8: np.uint64}[es]
    A = t.A.view(ut).reshape(X, Y, Z)
    yn = Y // npes
    assert np.array_equal(got.view(ut), np.stack([A[:, q * yn:(q + 1) * yn, :].reshape(-1) for q in range(npes)]))
    w.alltoalls(s, d, sps, dps, sbs, dbs, block, nblocks)              # the inverse exchange restores the x-slabs
    w.quiet(0)
    assert np.array_equal(w.view(s, sb).cpu().numpy(), t.A)


@pytest.mark.parametrize("npes,block,nblocks,sbs,sps,dbs,dps,soff,doff", [
    (5, 8, 4, 16, 64, 24, 96, 0, 0),            # alltoalls element form, 8-byte elements (dst = 3, sst = 2, nelems = 4)
    (7, 4, 9, 4, 36, 12, 108, 4, 8),            # 4-byte elements
    (4, 16, 3, 48, 200, 16, 48, 16, 32),        # 16-byte elements
    (6, 1000, 3, 1100, 4000, 1000, 3000, 3, 5),  # odd sizes and offsets: register path
    (3, 40000, 2, 40016, 90000, 40000, 80000, 0, 16),   # bulk path with a ragged last chunk
    (9, 1, 5, 2, 11, 1, 5, 1, 2),               # single bytes
])
def test_alltoalls_shapes_match_oracle(npes, block, nblocks, sbs, sps, dbs, dps, soff, doff):
    sspan = (npes - 1) * sps + (nblocks - 1) * sbs + block
    dspan = (npes - 1) * dps + (nblocks - 1) * dbs + block
    w, ow = _pair(npes, sspan + dspan + 8192)
    s, d = w.malloc(sspan + 64) + soff, w.malloc(dspan + 64) + doff
    os_, od = ow.malloc(sspan + 64) + soff, ow.malloc(dspan + 64) + doff
    pay = np.ascontiguousarray(gen.u64(npes * (sspan // 8 + 1), 21).view(np.uint8).reshape(npes, -1)[:, :sspan])
    w.view(s, sspan).copy_(torch.from_numpy(pay)); ow.view(os_, sspan)[:] = pay
    w.view(d, dspan).fill_(0xEE); ow.view(od, dspan)[:] = 0xEE
    w.alltoalls(d, s, dps, sps, dbs, sbs, block, nblocks); ow.alltoalls(od, os_, dps, sps, dbs, sbs, block, nblocks)
    w.quiet(0)
    assert np.array_equal(w.view(d, dspan).cpu().numpy(), ow.view(od, dspan))           # gaps between blocks untouched
    assert np.array_equal(w.view(s, sspan).cpu().numpy(), pay)


def test_alltoalls_argument_checks():
    w = World(4, 1 << 16, DEV)
    a, b = w.malloc(8192), w.malloc(8192)
    for args, code in [((b, a, 1 << 20, 64, 64, 64, 64, 1), ERR.RANGE),
                       ((a + 64, a, 64, 64, 64, 64, 64, 1), ERR.OVERLAP),
                       ((b, a, 256, 256, 32, 64, 64, 4), ERR.OVERLAP),          # dst_block_stride < block
                       ((b, a, 32, 256, 64, 64, 64, 1), ERR.OVERLAP)]:         # dst_pe_stride < block
        with pytest.raises(ShmemgError) as e:
            w.alltoalls(*args)
        assert e.value.code == code, (args, e.value)
    w.alltoalls(b, a, 64, 64, 64, 64, 0, 5)                                  # nothing to move
    with pytest.raises(ShmemgError) as e:
        w.ibput(b, a, 8, 64, 64, 3, 0, 1)                                    # ibput: destination blocks would overlap
    assert e.value.code == ERR.OVERLAP


def test_two_space_model_put_get_between_spaces():
    """a GPU space and a CPU space; capability query reports the CPU heap once attached; put / get between any
    two spaces match the oracle's slice assignments; CPU-space pointers are dereferenceable on the host."""
    npes, gb, cb, n = 4, 1 << 20, 1 << 19, 200000
    w, ow = _pair(npes, gb)
    assert not w.query_capabilities(TEAM.WORLD) & CAP.CPU_HEAP_PRESENT
    with pytest.raises(ShmemgError):
        w.cpu_malloc(64)                                                     # no CPU space yet
    w.cpu_heap_attach(cb); ow.attach_cpu_space(cb)
    assert w.query_capabilities(TEAM.WORLD) & CAP.CPU_HEAP_PRESENT and w.query_capabilities(TEAM.DEVICE_WORLD) & CAP.CPU_HEAP_PRESENT
    g, c = w.malloc(n), w.cpu_malloc(n)
    og, oc = ow.malloc(n), ow.cpu_malloc(n)
    assert (g, c) == (og, oc) and w.cpu_malloc(100) == ow.cpu_malloc(100)    # same allocation order -> same offsets
    pg = np.ascontiguousarray(gen.u64(npes * (n // 8 + 1), 31).view(np.uint8).reshape(npes, -1)[:, :n])
    pc = np.ascontiguousarray(gen.u64(npes * (n // 8 + 1), 32).view(np.uint8).reshape(npes, -1)[:, :n])
    w.view(g, n).copy_(torch.from_numpy(pg)); ow.view(og, n)[:] = pg
    w.cpu_view(c, n).copy_(torch.from_numpy(pc)); ow.cpu_view(oc, n)[:] = pc
    G, Cc = 0, 1
    for ds, do, ss, so, nb, pe, tg, put in [(Cc, 10, G, 3, 50000, 0, 2, True), (G, 1000, Cc, 7, 33333, 1, 0, False),
                                             (Cc, 60000, Cc, 0, 1000, 2, 1, True), (G, 90000, G, 0, 6400, 1, 3, True),
                                             (G, 150001, Cc, 99999, 12345, 3, 3, False), (Cc, 199000, G, 199000, 1000, 3, 0, True)]:
        (w.put_space if put else w.get_space)(ds, (c if ds else g) + do, ss, (c if ss else g) + so, nb, pe, tg)
        (ow.put_space if put else ow.get_space)(ds, (oc if ds else og) + do, ss, (oc if ss else og) + so, nb, pe, tg)
        w.quiet(0)                                                           # host visibility of the CPU space
    assert np.array_equal(w.view(g, n).cpu().numpy(), ow.view(og, n))
    assert np.array_equal(w.cpu_view(c, n).numpy(), ow.cpu_view(oc, n))
    import ctypes
    p = w.cpu_ptr(c + 5, 2)
    assert p and ctypes.string_at(p, 16) == ow.cpu_view(oc, n)[2, 5:21].tobytes()
    assert w.cpu_ptr(cb + 1, 0) == 0 and w.cpu_ptr(0, npes) == 0
    with pytest.raises(ShmemgError) as e:
        w.put_space(Cc, cb - 10, G, g, 64, 0, 1)
    assert e.value.code == ERR.RANGE
    w.cpu_free(c)
    assert w.cpu_malloc(n) == c
