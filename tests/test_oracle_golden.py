"""Regression of the oracle against tests/golden/cfg0_oracle.json (written by
tests/golden/make_golden.py from the oracle alone)."""
import json
import os

import pytest

from golden.make_golden import summary


def test_cfg0_oracle_regression():
    path = os.path.join(os.path.dirname(__file__), "golden", "cfg0_oracle.json")
    with open(path) as f:
        gold = json.load(f)
    now = summary()
    assert set(now) == set(gold)
    for t, g in gold.items():
        n = now[t]
        for k in ("survivors", "M", "cull_hist", "contributed"):
            assert n[k] == g[k], (t, k)
        for k in ("rgb_sum", "depth_sum", "alpha_sum"):
            assert n[k] == pytest.approx(g[k], rel=1e-11), (t, k)
        assert n["pixel_40_60"] == pytest.approx(g["pixel_40_60"], rel=1e-11)
