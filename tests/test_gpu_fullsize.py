"""Parity at BASELINE.json's full sizes, in the launch configuration bench.py times (defaults).

The oracle's 64-bit state digest after every `stride`-th step of the full run is stored in
tests/golden/trace_<cfg>.json (written by tests/golden/make_golden.py, which calls only oracle/).
A digest is a function of the whole state (id, edge, lane, bits(x), bits(v) of every ACTIVE vehicle
plus the counters), and the system is chaotic, so equality at the sampled steps means the
trajectories are the same.  The CUDA path must reproduce every stored digest, the ACTIVE count
at those steps, the final counts and the total number of vehicle-updates."""
import json
import os

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def _trace(name):
    path = os.path.join(GOLDEN, f"trace_{name}.json")
    if not os.path.exists(path):
        path = os.path.join(GOLDEN, f"trace_{name}_partial.json")      # prefix of a run still going
    if not os.path.exists(path):
        pytest.skip(f"{path} not generated yet (tests/golden/make_golden.py {name})")
    return json.load(open(path))


@pytest.mark.parametrize("name", ["cfg1", "cfg2", "cfg3", "cfg5", "cfg4"])
def test_full_run_matches_golden_digests(name):
    import paper_1807_01148_b200 as pkg
    from paper_1807_01148_b200 import workload as W
    tr = _trace(name)
    b = W.by_name(name)
    assert W.bundle_sha256(b) == tr["sha256"], "the seeded generator produced different inputs on this machine"
    sim = pkg.Sim(b, "cuda:0")
    done = 0
    for mark, want, active in zip(tr["marks"], tr["digests"], tr["active"]):
        if mark - done > 1:
            sim.step(mark - done - 1)
        got = int(sim.step_digest(1)[0])
        assert f"{got:016x}" == want, f"{name}: digest differs at step {mark}"
        done = mark
    st = sim.read_counts()
    assert st["step"] == tr["marks"][-1]
    if tr.get("complete", True):
        assert st["step"] == tr["steps"]
    # counters of the stored trace are those at its last mark (the whole run, or the prefix of an
    # oracle run that was still going when the file was committed: see make_golden.py)
    for key in ("n_pending", "n_active", "n_arrived"):
        assert st[key] == tr["final"][key], key
    assert st["vehicle_updates"] == tr["counters"]["updates"]
    if "edge_stats" in tr:                  # A11 and the edge counters: not covered by the digests
        es = sim.read_edge_stats()
        w = np.arange(1, len(es["entered"]) + 1, dtype=np.uint64)
        assert int(es["n_samples"]) == tr["edge_stats"]["n_samples"]
        for key, pair in tr["edge_stats"].items():
            if key == "n_samples":
                continue
            total, weighted = pair
            v = np.asarray(es[key], np.uint64)
            assert int(v.sum()) == total, key
            assert int((v * w).sum() & np.uint64(0xFFFFFFFFFFFFFFFF)) == weighted, key
    if "final_state" in tr:                 # every vehicle's final record, PENDING and ARRIVED ones included
        import importlib.util
        spec = importlib.util.spec_from_file_location("make_golden", os.path.join(GOLDEN, "make_golden.py"))
        mg = importlib.util.module_from_spec(spec)
        spec.loader.exec_module(mg)
        got_state = mg.state_checksums(sim.read_state())
        for key, pair in tr["final_state"].items():
            assert got_state[key] == pair, f"final {key}"
    assert np.all(np.diff(tr["marks"]) > 0)
    sim.close()


@pytest.mark.parametrize("name", ["cfg1", "cfg2", "cfg5", "cfg3"])
def test_full_run_emission_totals(name):
    """Section 6.3.4 at full size, default launch configuration, WHOLE run: the
    oracle's per-vehicle CO and fuel totals are stored as checksums of their fp32 bit patterns
    (tests/golden/emissions_<cfg>.json, written by make_golden.py --emissions from oracle/ only)."""
    import paper_1807_01148_b200 as pkg
    from paper_1807_01148_b200 import workload as W
    path = os.path.join(GOLDEN, f"emissions_{name}.json")
    if not os.path.exists(path):
        pytest.skip(f"{path} not generated yet (tests/golden/make_golden.py --emissions {name})")
    tr = json.load(open(path))
    b = W.by_name(name)
    assert W.bundle_sha256(b) == tr["sha256"]
    sim = pkg.Sim(dict(b, params=dict(b["params"], emissions=1)), "cuda:0")
    sim.step(tr["steps"] - 1)
    assert f"{int(sim.step_digest(1)[0]):016x}" == tr["final_digest"]
    assert sim.read_counts()["vehicle_updates"] == tr["updates"]
    em = sim.read_emissions()
    for key in ("co_g", "fuel_ml"):
        u = em[key].view(np.uint32).astype(np.uint64)
        w = np.arange(1, len(u) + 1, dtype=np.uint64)
        assert int(u.sum()) == tr[key]["bits_sum"], key
        assert int((u * w).sum() & np.uint64(0xFFFFFFFFFFFFFFFF)) == tr[key]["bits_weighted"], key
        assert float(em[key].astype(np.float64).sum()) == tr[key]["sum"], key
    sim.close()
