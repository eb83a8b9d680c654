"""Regression freeze of the oracle's trajectory (values written by tests/golden/make_oracle_golden.py, oracle only)."""
import importlib.util
import json
import os

import pytest

HERE = os.path.dirname(os.path.abspath(__file__))
spec = importlib.util.spec_from_file_location("make_oracle_golden", os.path.join(HERE, "golden", "make_oracle_golden.py"))
mk = importlib.util.module_from_spec(spec)
spec.loader.exec_module(mk)
GOLD = json.load(open(os.path.join(HERE, "golden", "oracle_golden.json")))


@pytest.mark.parametrize("name", sorted(mk.CASES))
def test_oracle_trajectory_frozen(name):
    got = mk.run(name)
    assert got["counters"] == GOLD[name]["counters"]
    assert got["header_t3"] == GOLD[name]["header_t3"]
    # positions are single-fmaf translations (bit-stable); quaternions go through libm sin/cos
    assert got["pos_sha256"] == GOLD[name]["pos_sha256"]
