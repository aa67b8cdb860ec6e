"""Seeded synthetic workloads shaped like BASELINE.json's five configs.

Inputs only: sizes, seeds, distributions, op lists.  No method arithmetic lives here.
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np

from . import gen
from .spec import CMP_GE, Program


# ------------------------------------------------------------------------------------------------
# C1: random non-fetching atomic adds
# ------------------------------------------------------------------------------------------------
@dataclass
class AtomicAddWorkload:
    npes: int
    nelem: int
    tgt_pe: np.ndarray   # int32 [n]
    idx: np.ndarray      # uint64 [n]
    val: np.ndarray      # int64 [n]


def c1_atomic_add(n_ops: int = 65536, npes: int = 4, nelem: int = 16384, seed: int = 0) -> AtomicAddWorkload:
    """tgt_pe uniform {0..npes-1}, idx uniform {0..nelem-1}, val uniform {1..1000} (config 1)."""
    return AtomicAddWorkload(
        npes, nelem,
        gen.uniform_i32(n_ops, 0, npes - 1, seed, stream=0),
        gen.uniform_i64(n_ops, 0, nelem - 1, seed, stream=1).astype(np.uint64),
        gen.uniform_i64(n_ops, 1, 1000, seed, stream=2))


# ------------------------------------------------------------------------------------------------
# C2: halo exchange on a (2B)^3 grid split 2x2x2, periodic (readings 21-23)
# ------------------------------------------------------------------------------------------------
class Halo:
    """Geometry and per-round op lists of the 2x2x2 periodic halo exchange.

    PE p has coordinates (px, py, pz) with p = (px*2 + py)*2 + pz and owns a B^3 block of fp64.
    Face f = 2*axis + dir (dir 0 = low side, 1 = high side).  Face f of p goes to the neighbour in
    direction `dir` along `axis`, where it lands in ghost slot f' = 2*axis + (1-dir), buffer
    `round & 1`; signal word sig[f'] is SET to the round number; the receiver waits `GE round`.
    """

    def __init__(self, B: int, seed: int = 1):
        self.B, self.seed, self.npes = int(B), int(seed), 8
        self.face_bytes = B * B * 8

    @staticmethod
    def coord(p: int):
        return (p >> 2) & 1, (p >> 1) & 1, p & 1

    @staticmethod
    def neighbour(p: int, axis: int, dir: int) -> int:      # periodic, 2 PEs per axis
        return p ^ (4 >> axis)

    def initial_U(self) -> np.ndarray:
        """[8, B^3] fp64 uniform [0,1): element (p, local c) is drawn at its GLOBAL grid index."""
        B, G = self.B, 2 * self.B
        flat = gen.uniform_f64(G ** 3, self.seed, stream=1000).reshape(G, G, G)
        out = np.empty((8, B ** 3), dtype=np.float64)
        for p in range(8):
            px, py, pz = self.coord(p)
            out[p] = flat[px * B:(px + 1) * B, py * B:(py + 1) * B, pz * B:(pz + 1) * B].reshape(-1)
        return out

    def program(self, with_consume: bool, with_U: bool = True) -> Program:
        prog = Program(8)
        fb = self.face_bytes
        if with_U:
            prog.obj("U", self.B ** 3 * 8, self.initial_U())
        prog.obj("send", 6 * fb)
        prog.obj("ghost", 2 * 6 * fb)
        prog.obj("sig", 6 * 8)
        if with_consume:
            prog.obj("consumed", 6 * fb)
        return prog

    def round_ops(self, prog: Program, rnd: int, with_consume: bool) -> Program:
        """One exchange round (rnd >= 1): 48 PUT_SIGNAL, 48 WAIT_UNTIL [, 48 local GETs of the ghosts]."""
        q = prog.fork()
        fb = self.face_bytes
        par = rnd & 1
        for p in range(8):
            for f in range(6):
                axis, d = f >> 1, f & 1
                t = self.neighbour(p, axis, d)
                fr = 2 * axis + (1 - d)
                q.put_signal(p, t, ("ghost", (par * 6 + fr) * fb), ("send", f * fb), fb, ("sig", fr * 8), rnd)
        for p in range(8):
            for fr in range(6):
                q.signal_wait_until(p, ("sig", fr * 8), CMP_GE, rnd)
        if with_consume:
            for p in range(8):
                for fr in range(6):
                    q.get(p, p, ("consumed", fr * fb), ("ghost", (par * 6 + fr) * fb), fb)
        return q


# ------------------------------------------------------------------------------------------------
# C3: MoE-style alltoall (uniform) and Zipf-skewed put batch
# ------------------------------------------------------------------------------------------------
def c3a_payload(npes: int = 64, block_bytes: int = 65536, seed: int = 2) -> np.ndarray:
    """[npes, npes*block_bytes] uint8 holding bf16 N(0,1) bit patterns (config 3)."""
    n16 = npes * npes * block_bytes // 2
    return gen.normal_bf16_bits(n16, seed, stream=0).view(np.uint8).reshape(npes, npes * block_bytes)


def c3a_put_program(npes: int = 64, block_bytes: int = 65536, seed: int = 2, payload=None) -> Program:
    """Uniform alltoall expressed as npes^2 puts + barrier (PE i sends block j to PE j's slot i)."""
    prog = Program(npes)
    prog.obj("src", npes * block_bytes, c3a_payload(npes, block_bytes, seed) if payload is None else payload)
    prog.obj("dst", npes * block_bytes)
    for i in range(npes):
        for j in range(npes):
            prog.put(i, j, ("dst", i * block_bytes), ("src", j * block_bytes), block_bytes)
    prog.barrier_all()
    return prog


@dataclass
class SkewedAlltoall:
    sizes: np.ndarray      # int64 [npes, npes] bytes, sizes[i, j] = bytes PE i sends to PE j
    src_off: np.ndarray    # exclusive prefix over j of row i
    dst_off: np.ndarray    # dst_off[i, j] = offset on PE j where PE i's block lands (prefix over i)
    src_bytes: int
    dst_bytes: int
    prog: Program


def c3b_skewed(npes: int = 64, unit: int = 4096, kmax: int = 64, s: float = 1.1, seed: int = 2,
               odd: bool = False) -> SkewedAlltoall:
    """Zipf(s) block sizes k*unit, k in 1..kmax (reading 17); offsets are exclusive prefix sums
    (reading 16).  `odd=True` perturbs sizes to odd byte counts for the alignment tests."""
    k = gen.zipf_ranks(npes * npes, s, kmax, seed, stream=1).reshape(npes, npes)
    sizes = k * unit
    if odd:
        sizes = sizes - gen.uniform_i64(npes * npes, 0, min(unit - 1, 61), seed, stream=2).reshape(npes, npes)
    src_off = np.cumsum(sizes, axis=1) - sizes
    dst_off = np.cumsum(sizes, axis=0) - sizes
    src_bytes = int(sizes.sum(axis=1).max())
    dst_bytes = int(sizes.sum(axis=0).max())
    prog = Program(npes)
    payload = gen.normal_bf16_bits(npes * ((src_bytes + 1) // 2), seed, stream=3).view(np.uint8)
    payload = payload.reshape(npes, -1)[:, :src_bytes]
    prog.obj("src", src_bytes, np.ascontiguousarray(payload))
    prog.obj("dst", dst_bytes)
    for i in range(npes):
        for j in range(npes):
            prog.put(i, j, ("dst", int(dst_off[i, j])), ("src", int(src_off[i, j])), int(sizes[i, j]))
    prog.barrier_all()
    return SkewedAlltoall(sizes, src_off, dst_off, src_bytes, dst_bytes, prog)


# ------------------------------------------------------------------------------------------------
# C4: RMAT fine-grained graph updates
# ------------------------------------------------------------------------------------------------
@dataclass
class GraphWorkload:
    npes: int
    scale: int
    verts_per_pe: int
    u: np.ndarray          # uint32 [E] source endpoint (global id)
    v: np.ndarray          # uint32 [E] destination endpoint (global id)

    def owner(self, x):
        return (x // self.verts_per_pe).astype(np.int32)

    def local(self, x):
        return (x % self.verts_per_pe).astype(np.uint64)


def c4_graph(scale: int = 22, edge_factor: int = 16, npes: int = 32, seed: int = 3) -> GraphWorkload:
    """RMAT (a,b,c,d) = (.57,.19,.19,.05); vertices block-partitioned: owner(x) = x // (2^scale/npes)."""
    n_edges = edge_factor << scale
    u, v = gen.rmat_edges(n_edges, scale, seed=seed)
    return GraphWorkload(npes, scale, (1 << scale) // npes, u, v)


# ------------------------------------------------------------------------------------------------
# C5: collectives
# ------------------------------------------------------------------------------------------------
def c5_f32(npes: int = 128, nelem: int = 1 << 20, seed: int = 4) -> np.ndarray:
    return gen.normal_f32(npes * nelem, seed, stream=0).reshape(npes, nelem)


def c5_i64(npes: int = 128, nelem: int = 1 << 19, seed: int = 4) -> np.ndarray:
    return gen.uniform_i64(npes * nelem, -(1 << 20), 1 << 20, seed, stream=1).reshape(npes, nelem)


def c5_fcollect_src(npes: int = 128, nbytes: int = 32768, seed: int = 4) -> np.ndarray:
    return gen.u64(npes * nbytes // 8, seed, stream=2).view(np.uint8).reshape(npes, nbytes)


# ------------------------------------------------------------------------------------------------
# NEXT-4 (i): FFT-style transpose ("FFT-driven spectral phases, many-to-many exchanges")
# ------------------------------------------------------------------------------------------------
@dataclass
class FftTranspose:
    """Slab transpose of a global array A[X][Y][Z] of `es`-byte elements (complex64: es = 8) over npes PEs: PE p holds the x-slab
    A[p*X/N : (p+1)*X/N, :, :]; afterwards PE q holds the y-slab B[x][yl][z] = A[x][q*Y/N + yl][z] (all x, x-major).  Seen as a
    block-strided alltoall: PE i sends to PE j, for each of its X/N local x, the contiguous chunk of Y/N rows."""
    npes: int
    X: int
    Y: int
    Z: int
    es: int
    A: np.ndarray                 # uint8 [npes, X/N * Y * Z * es]: the x-slabs

    @property
    def slab_bytes(self):
        return self.X // self.npes * self.Y * self.Z * self.es

    def params(self):
        """(block_bytes, nblocks, src_block_stride, src_pe_stride, dst_block_stride, dst_pe_stride) of the alltoalls call."""
        yn, xn = self.Y // self.npes, self.X // self.npes
        block = yn * self.Z * self.es
        return block, xn, self.Y * self.Z * self.es, block, block, xn * block


def fft_transpose(npes: int = 64, X: int = 1024, Y: int = 1024, Z: int = 256, es: int = 8, seed: int = 5) -> FftTranspose:
    assert X % npes == 0 and Y % npes == 0
    n = X * Y * Z * es
    A = gen.normal_f32(n // 4, seed, stream=0).view(np.uint8).reshape(npes, n // npes)        # complex64 = two N(0,1) floats
    return FftTranspose(npes, X, Y, Z, es, A)
