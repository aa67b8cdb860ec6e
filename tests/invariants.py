"""Schedule-independent checks for outputs that legitimately differ between legal schedules
(SURVEY.md 8(c) comparison table).  Applied to the oracle's outputs (CPU tests) and to the CUDA path's
outputs (GPU tests); they import neither."""
from __future__ import annotations

import numpy as np


def check_fetch_add(key: np.ndarray, val: np.ndarray, fetched: np.ndarray, init: np.ndarray,
                    final: np.ndarray) -> None:
    """key[i] = dense id of the target word of op i; val > 0 (no wraparound in the tested ranges).
    Per word: sorted by fetched value f, f(0) = init and f(j+1) = f(j) + v(j) -- the fetched values are
    the prefix sums of some permutation of the word's ops -- and final = init + sum v."""
    key = np.asarray(key, dtype=np.int64)
    val = np.asarray(val).astype(np.uint64)
    fetched = np.asarray(fetched).astype(np.uint64)
    init = np.asarray(init).astype(np.uint64)
    final = np.asarray(final).astype(np.uint64)
    assert (val > 0).all()
    order = np.lexsort((fetched, key))
    k, f, v = key[order], fetched[order], val[order]
    first = np.ones(len(k), dtype=bool)
    first[1:] = k[1:] != k[:-1]
    assert np.array_equal(f[first], init[k[first]]), "smallest fetched value of a word is not its initial value"
    cont = ~first
    assert np.array_equal(f[cont], (f[:-1] + v[:-1])[cont[1:]]), "fetched values are not prefix sums of a permutation"
    last = np.ones(len(k), dtype=bool)
    last[:-1] = k[1:] != k[:-1]
    exp_final = init.copy()
    exp_final[k[last]] = f[last] + v[last]
    assert np.array_equal(final, exp_final), "final word != init + sum of values"


def check_compare_swap_claim(key: np.ndarray, val: np.ndarray, fetched: np.ndarray, final: np.ndarray,
                             empty: int = 0xFFFFFFFFFFFFFFFF) -> None:
    """All ops are CAS(empty -> val) on slots initialised to `empty`, val != empty.  Per touched slot:
    exactly one op fetched `empty`, the slot's final value is that op's value, every other op fetched
    exactly the final value; untouched slots still hold `empty`."""
    key = np.asarray(key, dtype=np.int64)
    val = np.asarray(val).astype(np.uint64)
    fetched = np.asarray(fetched).astype(np.uint64)
    final = np.asarray(final).astype(np.uint64)
    e = np.uint64(empty)
    assert (val != e).all()
    won = fetched == e
    nwin = np.bincount(key[won], minlength=len(final))
    touched = np.bincount(key, minlength=len(final)) > 0
    assert np.array_equal(nwin[touched], np.ones(int(touched.sum()), dtype=nwin.dtype)), "slot not claimed exactly once"
    assert (nwin[~touched] == 0).all()
    assert (final[~touched] == e).all(), "untouched slot modified"
    assert np.array_equal(final[key[won]], val[won]), "final slot value is not the winner's value"
    assert np.array_equal(fetched[~won], final[key[~won]]), "a losing op fetched something other than the final value"
