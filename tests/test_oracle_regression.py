"""The oracle's outputs on small seeded batches have not changed (digests written by tests/golden/make_golden.py)."""
import importlib.util
import json
import os

HERE = os.path.dirname(os.path.abspath(__file__))


def test_oracle_regression_digests():
    spec = importlib.util.spec_from_file_location("make_golden", os.path.join(HERE, "golden", "make_golden.py"))
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    with open(os.path.join(HERE, "golden", "oracle_regression.json")) as f:
        want = json.load(f)
    assert mod.compute() == want
