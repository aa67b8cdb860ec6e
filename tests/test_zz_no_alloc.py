"""The entry point for callers that cannot allocate device memory: shmemg_atomic_fetch_add_batch_static_on_stream.

Who that is: code that is handed a stream, the slab and its input / output pointers but no allocator (a plug-in or callback
inside someone else's runtime), a process whose GPU memory was all given to one pool at start-up (a later cudaMalloc fails),
or a pipeline where cudaMalloc's device-wide synchronisation is not acceptable.  For them the scratch of the hot-set fetch-add
kernels is a fixed 8 MiB array inside libshmemg.so instead of a buffer registered with shmemg_set_scratch, and the call is
limited to 2^22 ops.

This file checks that the new call returns what the existing caller-scratch path returns.  Fetched values of a fetch-add batch
are only fixed up to the order in which the ops of one word executed, so "the same" is taken the way the other fetch-add tests
take it: the final heap words bit-exact, and per word the SORTED fetched values identical (both must be the word's prefix
sums).  Two calls are made back to back on the same counters with different op streams, because the array is shared and keeps
the first call's contents: the second call must not be disturbed by them.

The file name sorts last on purpose: pytest -x stops at the first failure, so a failure here cannot hide another test.  It makes
no assumption about what ran before it (own worlds, own inputs), so it passes alone in a fresh process and at the end of the
suite."""
import numpy as np
import pytest
import torch

from paper_2607_08006_b200 import World
from paper_2607_08006_b200.binding import AMO_HOT_AGGREGATE, AMO_THEN_BARRIER, ERR, STATIC_MAX_OPS, ShmemgError
from invariants import check_fetch_add
from workloads import gen

pytestmark = pytest.mark.gpu
DEV = "cuda:0"
NPES, WORDS = 3, 5000


def _stream(n, seed, idx_dtype):
    """n ops skewed towards a few words (so that the sampling kernel finds hot words and the per-CTA lists are used)."""
    r = gen.u64(n, seed)
    key = ((r % np.uint64(NPES * WORDS)) >> (r >> np.uint64(60))).astype(np.int64)
    return key, (key // WORDS).astype(np.int32), (key % WORDS).astype(idx_dtype)


def _world():
    w = World(NPES, WORDS * 8 + 8192, DEV)
    w.malloc(256)                                            # the counters do not start at offset 0
    a = w.malloc(WORDS * 8)
    init = (gen.u64(NPES * WORDS, 177) >> np.uint64(2)).reshape(NPES, WORDS)
    w.view(a, WORDS * 8, torch.int64).copy_(torch.from_numpy(init.view(np.int64)))
    return w, a, init.reshape(-1)


def _words(w, a):
    return w.view(a, WORDS * 8, torch.int64).cpu().numpy().view(np.uint64).reshape(-1).copy()


def _sorted_per_word(key, fetched):
    o = np.lexsort((fetched, key))
    return key[o], fetched[o]


@pytest.mark.parametrize("idx_dtype", [np.uint32, np.int64])
def test_static_scratch_fetch_add_equals_caller_scratch_path_twice_in_a_row(idx_dtype):
    calls = [((1 << 20) + 5, 401, 7), ((1 << 21) + 1029, 402, 3)]          # (ops, seed, value): ragged sizes, two different streams
    w_new, a_new, init = _world()                            # world driven through the new entry point: no scratch registered
    w_old, a_old, _ = _world()                               # world driven through the existing path with caller-owned scratch
    w_old.set_scratch_for(max(c[0] for c in calls))
    before = init
    for n, seed, v in calls:
        key, tgt, idx = _stream(n, seed, idx_dtype)
        t, i = torch.from_numpy(tgt).to(DEV), torch.from_numpy(idx).to(DEV)
        f_new = torch.full((n,), -1, dtype=torch.int64, device=DEV)
        f_old = torch.full((n,), -1, dtype=torch.int64, device=DEV)
        path = w_new.atomic_fetch_add_batch_static(a_new, t, i, f_new, val_scalar=v)
        assert path == 1, "the hot-set kernels did not run on the built-in scratch"
        w_old.atomic_fetch_add_batch(a_old, t, i, f_old, val=None, val_scalar=v, flags=AMO_HOT_AGGREGATE)
        w_new.quiet(0)
        w_old.quiet(0)
        fin_new, fin_old = _words(w_new, a_new), _words(w_old, a_old)
        assert np.array_equal(fin_new, fin_old)                             # integer work: bit-exact
        fn, fo = f_new.cpu().numpy().view(np.uint64), f_old.cpu().numpy().view(np.uint64)
        k1, s1 = _sorted_per_word(key, fn)
        k2, s2 = _sorted_per_word(key, fo)
        assert np.array_equal(k1, k2) and np.array_equal(s1, s2)            # per word the same set of fetched values
        check_fetch_add(key, np.full(n, v, dtype=np.uint64), fn, before, fin_new)       # and they are the prefix sums
        before = fin_new


def test_static_scratch_small_call_and_then_barrier():
    """Below 2^20 ops the plain kernel runs (no scratch at all, path 0); SHMEMG_AMO_THEN_BARRIER bumps the barrier epoch."""
    w, a, init = _world()
    n = 4099
    key, tgt, idx = _stream(n, 403, np.uint32)
    f = torch.empty(n, dtype=torch.int64, device=DEV)
    e0 = w.barrier_epoch()
    assert w.atomic_fetch_add_batch_static(a, torch.from_numpy(tgt).to(DEV), torch.from_numpy(idx).to(DEV), f, val_scalar=5,
                                           flags=AMO_THEN_BARRIER) == 0
    w.quiet(0)
    assert w.barrier_epoch() == e0 + 1
    check_fetch_add(key, np.full(n, 5, dtype=np.uint64), f.cpu().numpy().view(np.uint64), init, _words(w, a))


def test_static_scratch_refuses_more_than_the_limit():
    """One op more than SHMEMG_STATIC_MAX_OPS: refused on the host with the reason in words; nothing is launched or written."""
    w, a, init = _world()
    n = STATIC_MAX_OPS + 1
    z = torch.zeros(n, dtype=torch.int32, device=DEV)
    f = torch.full((n,), -1, dtype=torch.int64, device=DEV)
    with pytest.raises(ShmemgError) as ei:
        w.atomic_fetch_add_batch_static(a, z, z, f, val_scalar=1)
    assert ei.value.code == ERR.NOMEM and "SHMEMG_STATIC_MAX_OPS" in str(ei.value) and str(n) in str(ei.value)
    with pytest.raises(ShmemgError) as ei:
        w.atomic_fetch_add_batch_static(a, z[:8], z[:8], f[:8], val_scalar=1, flags=1)      # WARP_AGGREGATE is not accepted here
    assert ei.value.code == ERR.ARG
    w.quiet(0)
    assert np.array_equal(_words(w, a), init) and bool((f == -1).all())
    # exactly the limit is accepted
    n = STATIC_MAX_OPS
    assert w.atomic_fetch_add_batch_static(a, z[:n], z[:n], f[:n], val_scalar=1) == 1
    w.quiet(0)
    fin = _words(w, a)
    assert fin[0] == init[0] + np.uint64(n) and np.array_equal(fin[1:], init[1:])
    assert np.array_equal(np.sort(f[:n].cpu().numpy().view(np.uint64)), init[0] + np.arange(n, dtype=np.uint64))
