"""Delay-depth tuning: host logic on CPU, one small measured run on GPU."""
import json

import pytest

from paper_2602_05255_b200 import tune


def test_heuristic_is_the_papers_rule():
    assert tune.heuristic_delay("det", 1280, 8) == 16      # n/10k
    assert tune.heuristic_delay("pf", 1280, 8) == 8        # n/20k
    assert tune.heuristic_delay("det", 32, 8) == 0


def test_recommended_delay_uses_the_table_then_the_rule(monkeypatch):
    monkeypatch.setattr(tune, "_TABLE", [
        {"kind": "det", "dtype": "f64", "n": 512, "k": 1, "best": 32},
        {"kind": "det", "dtype": "f64", "n": 128, "k": 2, "best": 0},
        {"kind": "pf", "dtype": "f64", "n": 128, "k": 1, "best": 0},
    ])
    assert tune.recommended_delay("det", 512, 1) == 32
    assert tune.recommended_delay("det", 600, 1) == 32           # nearest tuned shape
    assert tune.recommended_delay("det", 128, 2) == 0
    assert tune.recommended_delay("det", 8192, 8) == tune.heuristic_delay("det", 8192, 8)   # too far: rule
    assert tune.recommended_delay("det", 512, 1, cplx=True) == tune.heuristic_delay("det", 512, 1)
    assert tune.recommended_delay("pf", 128, 1) == 0


def test_committed_table_is_well_formed():
    tune._TABLE = None
    for e in tune.load_table():
        assert e["kind"] in ("det", "pf") and e["n"] > 0 and e["k"] > 0 and e["best"] >= 0
        assert e["best"] in [t["K"] for t in e["table"]]


@pytest.mark.gpu
def test_tune_delay_measures_every_depth():
    r = tune.tune_delay("det", 64, 2, W=512, depths=(0, 2, 4, 64), steps=6)
    ks = [t["K"] for t in r["table"]]
    assert ks == [0, 2, 4]                                       # K*k >= n is skipped (T < n/k)
    assert r["best"] in ks and all(t["walker_updates_per_s"] > 0 for t in r["table"])
    assert r["heuristic"] == 3
    json.dumps(r)
    r = tune.tune_delay("pf", 32, 1, W=256, depths=(0, 2), steps=6, mode="forced")
    assert [t["K"] for t in r["table"]] == [0, 2]
