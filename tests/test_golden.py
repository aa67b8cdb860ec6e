"""The oracle still produces the stored checksums of tests/golden/oracle_checksums.txt (written by
tests/golden/make_golden.py from oracle/ only).  CPU only."""
import importlib.util
import os

HERE = os.path.dirname(os.path.abspath(__file__))


def test_oracle_reproduces_stored_checksums():
    spec = importlib.util.spec_from_file_location("make_golden", os.path.join(HERE, "golden", "make_golden.py"))
    mg = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mg)
    stored = dict(ln.split() for ln in open(os.path.join(HERE, "golden", "oracle_checksums.txt")) if ln.strip() and ln[0] != "#")
    now = dict(mg.cases())
    assert now == stored
