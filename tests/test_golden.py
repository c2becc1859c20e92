"""The oracle reproduces its stored stage counts and checksums (tests/golden/oracle_counts.txt, written by
tests/golden/make_golden.py from datagen/ + oracle/ only).  The paper prints no worked example to store instead."""
import importlib.util
import os

HERE = os.path.dirname(os.path.abspath(__file__))


def test_oracle_matches_its_golden_counts():
    spec = importlib.util.spec_from_file_location("make_golden", os.path.join(HERE, "golden", "make_golden.py"))
    mg = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mg)
    stored = open(os.path.join(HERE, "golden", "oracle_counts.txt")).read().strip().splitlines()
    assert stored == mg.lines()
