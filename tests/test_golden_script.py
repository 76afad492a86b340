"""The script that writes the stored oracle traces (tests/golden/make_golden.py) runs on the CPU
only and produces what the full-size GPU test reads; the committed traces are consistent."""
import importlib.util
import json
import os

import numpy as np

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def _load_script():
    spec = importlib.util.spec_from_file_location("make_golden", os.path.join(GOLDEN, "make_golden.py"))
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    return mod


def test_script_reproduces_the_committed_config1_trace(tmp_path, monkeypatch):
    mod = _load_script()
    monkeypatch.setattr(mod, "HERE", str(tmp_path))
    mod.run("cfg1", 600)
    new = json.load(open(tmp_path / "trace_cfg1.json"))
    old = json.load(open(os.path.join(GOLDEN, "trace_cfg1.json")))
    for key in ("sha256", "steps", "marks", "digests", "active", "counters", "final", "edge_stats", "final_state"):
        assert new[key] == old[key], key
    assert new["complete"] and new["marks"][-1] == new["steps"] == 3600
    assert new["final"] == dict(n_pending=0, n_active=0, n_arrived=500)


def test_committed_traces_are_well_formed():
    names = [f for f in os.listdir(GOLDEN) if f.startswith("trace_") and f.endswith(".json")]
    assert {"trace_cfg1.json", "trace_cfg2.json", "trace_cfg5.json"} <= set(names)
    for f in names:
        t = json.load(open(os.path.join(GOLDEN, f)))
        assert len(t["marks"]) == len(t["digests"]) == len(t["active"]) > 0, f
        assert (np.diff(t["marks"]) > 0).all() and t["marks"][-1] <= t["steps"], f
        assert all(len(d) == 16 for d in t["digests"]), f     # (a drained run repeats its last digest)
        assert t.get("complete", True) == (t["marks"][-1] == t["steps"]), f
        c = t["counters"]
        assert c["updates"] > 0 and c["departures"] >= c["arrivals"], f
        # one trace per config: a prefix file only where no complete one exists
        if f.endswith("_partial.json"):
            assert f.replace("_partial", "") not in names, f
