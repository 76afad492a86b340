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


def test_full_size_config3_rerouting_on_sampled_origins():
    """ts_reroute at the size the metric names (1 M vehicles, 4 096 origins, 62 M route entries), default
    launch configuration.  Inputs come from the workload alone: at step 0 nothing has left an edge, so the
    weights are the free-flow weights (reading R37).  Sampled outputs the oracle computes one by one: the
    trees of 10 origins drawn from a seed, and every route of the ~2 400 vehicles that start there, edge by
    edge.  Properties of ALL 1 M routes: same origin and destination, contiguous, never costlier than the
    route given, offsets consistent."""
    import paper_1807_01148_b200 as pkg
    from oracle import reroute as R
    from paper_1807_01148_b200 import workload as W
    b = W.by_name("cfg3")
    wf = W.free_flow_weights(b)
    ef, et = b["edge_from"].astype(np.int64), b["edge_to"].astype(np.int64)
    off, re = b["route_off"].astype(np.int64), b["route_edges"].astype(np.int64)
    origin, dest = ef[re[off[:-1]]], et[re[off[1:] - 1]]
    sim = pkg.Sim(dict(b, params=dict(b["params"], route_capacity=2 * len(re) + 4096)), "cuda:0")
    info = sim.reroute(wf)
    assert np.array_equal(info["w"], wf) and info["n_rerouted"] == b["n_vehicles"]
    assert info["n_trees"] == len(np.unique(origin))
    g_off, g_edges = sim.read_routes()
    sim.close()
    g_off, g_edges = g_off.astype(np.int64), g_edges.astype(np.int64)
    assert g_off[0] == 0 and g_off[-1] == len(g_edges) == info["route_entries"] and (np.diff(g_off) >= 1).all()
    # every route: origin, destination, contiguity, cost
    assert np.array_equal(ef[g_edges[g_off[:-1]]], origin) and np.array_equal(et[g_edges[g_off[1:] - 1]], dest)
    inner = np.ones(len(g_edges), bool)
    inner[g_off[1:-1] - 1] = False                       # last edge of every route but the final one
    inner[-1] = False
    idx = np.nonzero(inner)[0]
    assert (et[g_edges[idx]] == ef[g_edges[idx + 1]]).all()
    new_cost = np.add.reduceat(wf[g_edges].astype(np.int64), g_off[:-1])
    old_cost = np.add.reduceat(wf[re].astype(np.int64), off[:-1])
    assert (new_cost <= old_cost).all() and (new_cost < old_cost).any()
    # sampled origins against the oracle's trees
    rng = np.random.default_rng(20180701)
    src = np.sort(rng.choice(np.unique(origin), 10, replace=False))
    _, pred = R.shortest_path_trees(b["n_nodes"], b["edge_from"], b["edge_to"], wf, src)
    checked = 0
    for r, s in enumerate(src):
        for i in np.nonzero(origin == s)[0]:
            path, v = [], int(dest[i])
            while v != s:
                e = int(pred[r, v]); path.append(e); v = int(ef[e])
            assert g_edges[g_off[i]:g_off[i + 1]].tolist() == path[::-1], f"vehicle {i} from origin {s}"
            checked += 1
    assert checked > 1500


def test_full_size_config3_static_assignment_properties():
    """ts_sue_solve on config 3's network and demand (65 535 nodes, 987 650 OD pairs, one hour): properties that
    hold at any size -- flow conservation at every node, non-negative flows, an objective (Eq. 6) that never
    increases (PAPER.md:335 step 3), a relative gap that shrinks, BPR times (Eq. 3) recomputed from the flows."""
    import paper_1807_01148_b200 as pkg
    from paper_1807_01148_b200 import workload as W
    b = W.by_name("cfg3")
    inp = W.sue_inputs(b, horizon_s=3600.0)
    N, ef, et = b["n_nodes"], b["edge_from"].astype(np.int64), b["edge_to"].astype(np.int64)
    x, t, info = pkg.sue_solve(N, ef, et, inp["t0"], inp["cap"], inp["od_origin"], inp["od_dest"], inp["od_trips"], iterations=6)
    assert (x >= 0).all() and (np.diff(info["objective"]) <= 1e-9 * info["objective"][0]).all()
    assert info["gap"][-1] < 0.5 * info["gap"][0] and all(0.0 <= a <= 1.0 for a in info["step"])
    net = np.zeros(N)
    np.add.at(net, et, x); np.add.at(net, ef, -x)
    want = np.zeros(N)
    np.add.at(want, inp["od_dest"].astype(np.int64), inp["od_trips"].astype(float))
    np.add.at(want, inp["od_origin"].astype(np.int64), -inp["od_trips"].astype(float))
    assert np.allclose(net, want, atol=1e-6 * inp["od_trips"].sum())
    r = x / inp["cap"]
    assert np.allclose(t, inp["t0"] * (1.0 + 0.15 * r ** 4), rtol=1e-12)
    assert info["n_trees"] == 7 * len(np.unique(inp["od_origin"]))
