"""Pins of the NEXT-4 oracle routines (CPU only): the block-strided alltoall against numpy transposes of the GLOBAL array, the
contiguous alltoall and the OpenSHMEM alltoalls element form; the two-space put / get against numpy slice assignment."""
import numpy as np
import pytest

from oracle import oracle as orc
from workloads import configs, gen


def test_fft_transpose_equals_numpy_transpose_of_the_global_array_and_is_an_involution():
    t = configs.fft_transpose(npes=4, X=8, Y=12, Z=5, es=8, seed=7)
    N, xn, yn = t.npes, t.X // t.npes, t.Y // t.npes
    sb = t.slab_bytes
    w = orc.OracleWorld(N, 3 * sb + 1024)
    s, d, back = w.malloc(sb), w.malloc(sb), w.malloc(sb)
    w.view(s, sb)[:] = t.A
    block, nblocks, sbs, sps, dbs, dps = t.params()
    w.alltoalls(d, s, dps, sps, dbs, sbs, block, nblocks)
    A = t.A.view(np.uint64).reshape(t.X, t.Y, t.Z)                         # the global array (x-slabs concatenated)
    want = np.stack([A[:, q * yn:(q + 1) * yn, :].reshape(-1) for q in range(N)])     # y-slab of PE q, x-major
    assert np.array_equal(w.view(d, sb, np.uint64), want)
    # the inverse exchange (roles of the strides swapped) restores the x-slabs
    w.alltoalls(back, d, sps, dps, sbs, dbs, block, nblocks)
    assert np.array_equal(w.view(back, sb), t.A)
    # each destination byte is written exactly once: sizes match and nothing else in the heap changed
    assert np.array_equal(w.view(s, sb), t.A)


def test_alltoalls_reduces_to_alltoall_and_to_the_openshmem_element_form():
    N, n = 5, 24
    w = orc.OracleWorld(N, 8192)
    s, d1, d2 = w.malloc(N * n), w.malloc(N * n), w.malloc(N * n)
    w.view(s, N * n)[:] = gen.u64(N * N * n // 8, 3).view(np.uint8).reshape(N, N * n)
    w.alltoall(d1, s, n)
    w.alltoalls(d2, s, n, n, n, n, n, 1)                                   # one block of n bytes per PE pair
    assert np.array_equal(w.view(d1, N * n), w.view(d2, N * n))
    w.alltoalls(d2, s, n, n, 8, 8, 8, n // 8)                              # the same bytes as n/8 blocks of one element
    assert np.array_equal(w.view(d1, N * n), w.view(d2, N * n))
    # alltoalls(dest, source, dst = 3, sst = 2, nelems = 4) on 8-byte elements, against fancy indexing
    es, dst, sst, ne = 8, 3, 2, 4
    w2 = orc.OracleWorld(N, 1 << 14)
    s2, d2 = w2.malloc(N * ne * sst * es), w2.malloc(N * ne * dst * es)
    src = gen.u64(N * N * ne * sst, 4).reshape(N, N * ne * sst)
    w2.view(s2, N * ne * sst * es, np.uint64)[:] = src
    w2.view(d2, N * ne * dst * es, np.uint64)[:] = 0
    w2.alltoalls(d2, s2, ne * dst * es, ne * sst * es, dst * es, sst * es, es, ne)
    want = np.zeros((N, N * ne * dst), dtype=np.uint64)
    for i in range(N):
        for j in range(N):
            want[j, (i * ne + np.arange(ne)) * dst] = src[i, (j * ne + np.arange(ne)) * sst]
    assert np.array_equal(w2.view(d2, N * ne * dst * es, np.uint64), want)


def test_alltoalls_argument_checks():
    w = orc.OracleWorld(2, 1024)
    w.alltoalls(0, 512, 8, 8, 8, 8, 0, 3)                                  # nothing to move
    with pytest.raises(orc.OracleError):
        w.alltoalls(0, 512, 400, 8, 8, 8, 300, 1)                          # destination leaves the heap
    with pytest.raises(orc.OracleError):
        w.alltoalls(0, 16, 16, 16, 16, 16, 16, 1)                          # footprints overlap


def test_two_space_put_get_are_slice_assignments_between_two_heaps():
    rng = np.random.default_rng(5)
    N, gb, cb = 3, 4096, 2048
    w = orc.OracleWorld(N, gb)
    w.attach_cpu_space(cb)
    g, c = w.malloc(1000), w.cpu_malloc(1000)
    w.view(g, 1000)[:] = rng.integers(0, 256, (N, 1000), dtype=np.uint8)
    w.cpu_view(c, 1000)[:] = rng.integers(0, 256, (N, 1000), dtype=np.uint8)
    G, Cc = w.view(g, 1000).copy(), w.cpu_view(c, 1000).copy()
    w.put_space(1, c + 10, 0, g + 3, 500, pe=0, target=2)                  # GPU window of PE 0 -> CPU window of PE 2
    Cc[2, 10:510] = G[0, 3:503]
    w.get_space(0, g + 100, 1, c + 7, 333, pe=1, target=0)                 # CPU window of PE 0 -> GPU window of PE 1
    G[1, 100:433] = Cc[0, 7:340]
    w.put_space(1, c + 600, 1, c, 100, pe=2, target=1)                     # CPU -> CPU
    Cc[1, 600:700] = Cc[2, 0:100]
    w.put_space(0, g + 900, 0, g, 64, pe=1, target=1)                      # GPU -> GPU (= put)
    G[1, 900:964] = G[1, 0:64]
    assert np.array_equal(w.view(g, 1000), G) and np.array_equal(w.cpu_view(c, 1000), Cc)
    with pytest.raises(orc.OracleError):
        w.put_space(1, cb - 10, 0, g, 64, pe=0, target=1)                  # leaves the CPU window
