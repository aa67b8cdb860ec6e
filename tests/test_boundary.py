"""CPU-only checks of the boundary: the C-ABI library loads and exports every symbol the headers declare,
the binding's table matches the headers, and the product path does not touch oracle/."""
import ctypes
import os
import re

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    names = []
    for h in sorted(f for f in os.listdir(os.path.join(ROOT, "include")) if f.endswith(".h")):
        src = open(os.path.join(ROOT, "include", h)).read()
        src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
        names += re.findall(r"SHMEMG_API\s+[\w\s\*]+?\b(shmemg?_\w+)\s*\(", src)
    return names


def test_library_exports_every_declared_symbol():
    from paper_2607_08006_b200 import _build, binding
    _build.build()
    names = _declared()
    assert len(names) >= 35 and len(set(names)) == len(names)
    L = ctypes.CDLL(binding.LIB_PATH)
    for n in names:
        assert hasattr(L, n), "library does not export " + n
    assert set(names) == set(binding.SYMBOLS), set(names) ^ set(binding.SYMBOLS)
    binding.lib()


def test_descriptor_layout_matches_header():
    from paper_2607_08006_b200 import binding
    d = binding.OP_DTYPE
    assert d.itemsize == 64
    offs = {n: d.fields[n][1] for n in d.names}
    assert offs == {"opcode": 0, "sig_op": 1, "cmp": 2, "ctx": 3, "initiator_pe": 4, "target_pe": 8,
                    "reserved1": 12, "rem_off": 16, "loc_off": 24, "nbytes": 32, "value": 40, "cond": 48, "sig_off": 56}
    hdr = open(os.path.join(ROOT, "include", "shmemg.h")).read()
    for k, v in vars(binding.OP).items():
        if k.isupper():
            assert re.search(r"SHMEMG_OP_%s = %d\b" % (k, v), hdr), k
    for k, v in vars(binding.CAP).items():
        if k.isupper():
            assert re.search(r"SHMEMG_CAP_%s\s+\(1ull << %d\)" % (k, v.bit_length() - 1), hdr), k


def test_host_only_entry_points_without_gpu():
    """No compute: argument checking that needs no device."""
    from paper_2607_08006_b200 import binding
    L = binding.lib()
    assert L.shmemg_slab_bytes_required(0, 100) == 0
    CTL = 65536 + (4 << 20)                    # control region + plan arena
    assert L.shmemg_slab_bytes_required(4, 1000) == 4 * 1024 + CTL
    os.environ["SHMEMG_SYMMETRIC_SIZE"] = "2K"
    try:
        assert L.shmemg_slab_bytes_required(3, 0) == 3 * 2048 + CTL
    finally:
        del os.environ["SHMEMG_SYMMETRIC_SIZE"]
    assert L.shmemg_slab_bytes_required(3, 0) == 0
    out = ctypes.c_void_p()
    assert L.shmemg_init(0, 100, 1, 100, ctypes.byref(out)) == binding.ERR.ARG
    assert L.shmemg_n_pes(None) == binding.ERR.ARG
    assert L.shmemg_ptr(None, 0, 0) is None
    assert L.shmemg_batch_plan_bytes(None, None, 0) == 0
    assert L.shmemg_batch_work_bytes(None, 10, 0) == 0
    assert L.shmemg_enqueue_batch(None, None, 0, None) == binding.ERR.ARG


def test_product_path_never_imports_oracle():
    pkg = os.path.join(ROOT, "paper_2607_08006_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in src.replace("shares nothing with oracle/", ""), f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            src = open(os.path.join(ROOT, "oracle", f)).read()
            assert "paper_2607_08006_b200" not in src and "shmemg.h" not in src, f


def test_loader_translation_is_pure_marshalling():
    from paper_2607_08006_b200.binding import OP_DTYPE
    from paper_2607_08006_b200.loader import Loaded
    from workloads.spec import Program
    p = Program(2)
    p.obj("a", 64)
    p.obj("b", 64)
    p.put_signal(0, 1, ("b", 8), ("a", 16), 24, ("b", 56), 7, 1)
    fake = Loaded.__new__(Loaded)
    fake.off, fake.names = {"a": (512, 64), "b": (1024, 64)}, ["a", "b"]
    ops = fake.translate(p)
    assert ops.dtype == OP_DTYPE and len(ops) == 1
    o = ops[0]
    assert (o["opcode"], o["sig_op"], o["initiator_pe"], o["target_pe"]) == (3, 1, 0, 1)
    assert (o["rem_off"], o["loc_off"], o["sig_off"], o["nbytes"], o["value"]) == (1032, 528, 1080, 24, 7)
