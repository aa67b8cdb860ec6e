"""ctypes front-end of workloads/gen.c: seeded, counter-based input generators.

Shared by the CUDA-path harness and the oracle harness; holds no method arithmetic
(SURVEY.md Appendix D).  The C file is compiled on first use with the system gcc.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "gen.c")
_SO = os.path.join(_HERE, "_gen.so")
_lib = None


def build(force: bool = False) -> str:
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        tmp = _SO + ".tmp%d" % os.getpid()
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-shared", "-fPIC", "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _SO)
    return _SO


def _load():
    global _lib
    if _lib is None:
        lib = C.CDLL(build())
        u64, i64, u32, i32, vp = C.c_uint64, C.c_int64, C.c_uint32, C.c_int32, C.c_void_p
        lib.wl_mix64.restype = u64
        lib.wl_mix64.argtypes = [u64, u64, u64]
        lib.wl_fill_u64.argtypes = [vp, u64, u64, u64, u64]
        lib.wl_fill_uniform_i64.argtypes = [vp, u64, i64, u64, u64, u64, u64]
        lib.wl_fill_uniform_i32.argtypes = [vp, u64, i32, u32, u64, u64, u64]
        lib.wl_fill_uniform_f64.argtypes = [vp, u64, u64, u64, u64]
        lib.wl_fill_normal_f32.argtypes = [vp, u64, u64, u64, u64]
        lib.wl_fill_normal_bf16.argtypes = [vp, u64, u64, u64, u64]
        lib.wl_rmat_edges.argtypes = [vp, vp, u64, C.c_int, u32, u32, u32, u64, u64]
        for f in ("wl_fill_u64", "wl_fill_uniform_i64", "wl_fill_uniform_i32", "wl_fill_uniform_f64",
                  "wl_fill_normal_f32", "wl_fill_normal_bf16", "wl_rmat_edges"):
            getattr(lib, f).restype = None
        _lib = lib
    return _lib


def _p(a: np.ndarray):
    assert a.flags["C_CONTIGUOUS"]
    return a.ctypes.data


def mix64(seed: int, stream: int, i: int) -> int:
    return int(_load().wl_mix64(seed, stream, i))


def u64(n: int, seed: int, stream: int = 0, i0: int = 0) -> np.ndarray:
    out = np.empty(n, dtype=np.uint64)
    _load().wl_fill_u64(_p(out), n, seed, stream, i0)
    return out


def uniform_i64(n: int, lo: int, hi: int, seed: int, stream: int = 0, i0: int = 0) -> np.ndarray:
    """Uniform integers in the closed range [lo, hi]."""
    out = np.empty(n, dtype=np.int64)
    _load().wl_fill_uniform_i64(_p(out), n, lo, hi - lo + 1, seed, stream, i0)
    return out


def uniform_i32(n: int, lo: int, hi: int, seed: int, stream: int = 0, i0: int = 0) -> np.ndarray:
    out = np.empty(n, dtype=np.int32)
    _load().wl_fill_uniform_i32(_p(out), n, lo, hi - lo + 1, seed, stream, i0)
    return out


def uniform_f64(n: int, seed: int, stream: int = 0, i0: int = 0) -> np.ndarray:
    """Uniform [0,1): 53-bit integers times 2^-53."""
    out = np.empty(n, dtype=np.float64)
    _load().wl_fill_uniform_f64(_p(out), n, seed, stream, i0)
    return out


def normal_f32(n: int, seed: int, stream: int = 0, i0: int = 0) -> np.ndarray:
    out = np.empty(n, dtype=np.float32)
    _load().wl_fill_normal_f32(_p(out), n, seed, stream, i0)
    return out


def normal_bf16_bits(n: int, seed: int, stream: int = 0, i0: int = 0) -> np.ndarray:
    """N(0,1) rounded to bf16 (RNE); returned as uint16 bit patterns."""
    out = np.empty(n, dtype=np.uint16)
    _load().wl_fill_normal_bf16(_p(out), n, seed, stream, i0)
    return out


def rmat_edges(n_edges: int, scale: int, a: float = 0.57, b: float = 0.19, c: float = 0.19,
               seed: int = 3, e0: int = 0):
    """RMAT edge list as two uint32 arrays (u, v); d = 1-a-b-c. Integer thresholds, no noise."""
    ta = int(a * 2.0 ** 32)
    tab = int((a + b) * 2.0 ** 32)
    tabc = int((a + b + c) * 2.0 ** 32)
    u = np.empty(n_edges, dtype=np.uint32)
    v = np.empty(n_edges, dtype=np.uint32)
    _load().wl_rmat_edges(_p(u), _p(v), n_edges, scale, ta, tab, tabc, seed, e0)
    return u, v


def zipf_ranks(n: int, s: float, kmax: int, seed: int, stream: int = 0, i0: int = 0) -> np.ndarray:
    """Ranks k in 1..kmax with P(k) ~ k^-s, by inverse-CDF lookup of a uniform 64-bit draw."""
    w = np.arange(1, kmax + 1, dtype=np.float64) ** (-s)
    cdf = np.cumsum(w) / np.sum(w)
    cdf[-1] = 1.0
    r = (u64(n, seed, stream, i0) >> np.uint64(11)).astype(np.float64) * 2.0 ** -53
    return (np.searchsorted(cdf, r, side="right") + 1).clip(1, kmax).astype(np.int64)
