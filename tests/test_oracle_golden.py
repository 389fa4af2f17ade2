"""Regression guard: the fp32 oracle on config 1 still produces the committed digest
(tests/golden/c1_oracle_f32.txt, written by tests/golden/make_golden.py from oracle/ only)."""
import importlib.util
import os


def test_c1_oracle_digest_unchanged(oracle):
    here = os.path.join(os.path.dirname(__file__), "golden")
    spec = importlib.util.spec_from_file_location("make_golden", os.path.join(here, "make_golden.py"))
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    assert mod.digest() == open(os.path.join(here, "c1_oracle_f32.txt")).read()
