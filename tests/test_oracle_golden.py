"""Drift guard: the oracle still reproduces tests/golden/oracle_regression.json (written by tests/golden/make_golden.py
from the oracle alone; see tests/golden/README.md)."""
import importlib.util
import json
import os

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))


def test_oracle_reproduces_stored_values():
    spec = importlib.util.spec_from_file_location("make_golden", os.path.join(HERE, "golden", "make_golden.py"))
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    now = mod.build()
    with open(os.path.join(HERE, "golden", "oracle_regression.json")) as f:
        stored = json.load(f)
    assert sorted(now) == sorted(stored)
    for key in stored:
        a, b = np.asarray(now[key], dtype=np.float64), np.asarray(stored[key], dtype=np.float64)
        assert a.shape == b.shape, key
        assert np.allclose(a, b, rtol=0, atol=1e-11, equal_nan=True), key
