"""The seeded generator and the oracle still produce the frozen checksums (tests/golden/oracle_checksums.json,
written by tests/golden/make_golden.py from oracle/ only)."""
import importlib.util
import json
import os

HERE = os.path.dirname(os.path.abspath(__file__))


def test_oracle_checksums_unchanged():
    spec = importlib.util.spec_from_file_location("make_golden", os.path.join(HERE, "golden", "make_golden.py"))
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    with open(os.path.join(HERE, "golden", "oracle_checksums.json")) as fh:
        frozen = json.load(fh)
    assert mod.compute() == frozen
