"""Pins of the re-routing oracle (oracle/reroute.py; R37-R41) against
things other than itself: weights worked by hand, distances against Bellman-Ford written out here
and against SciPy's Floyd-Warshall, the tie-break against a brute-force enumeration of every
shortest path on tiny graphs, and the properties a re-routed demand must have."""
import itertools

import numpy as np
import pytest
import scipy.sparse as sp
from scipy.sparse.csgraph import floyd_warshall

from oracle import Oracle
from oracle import reroute as R
from paper_1807_01148_b200 import workload as W


def test_edge_weights_by_hand():
    """R37: round-half-up(256 * sum / exited); free-flow weight where nothing left the edge; clamps."""
    exited = np.array([3, 0, 1, 2, 1, 7])
    ssum = np.array([10, 999, 0, 5, 1 << 30, 7 * 41])
    wfree = np.array([11, 22, 33, 44, 55, 66])
    got = R.edge_weights(exited, ssum, wfree)
    #  10/3 steps = 853.33 -> 853;  free-flow;  0 -> clamped to 1;  2.5 steps = 640;  clamp 2^20;  41 steps
    assert got.tolist() == [853, 22, 1, 640, 1 << 20, 41 * 256]
    assert R.edge_weights([2], [1], [9]).tolist() == [128]            # 0.5 step
    assert R.edge_weights([3], [1], [9]).tolist() == [85]             # 85.33
    assert R.edge_weights([3], [2], [9]).tolist() == [171]            # 170.67 -> 171
    assert R.edge_weights([2], [3], [9]).tolist() == [384]


def _bellman_ford(n, ef, et, w, s):
    d = [float("inf")] * n
    d[s] = 0
    for _ in range(n):
        for e in range(len(ef)):
            if d[ef[e]] + w[e] < d[et[e]]:
                d[et[e]] = d[ef[e]] + w[e]
    return d


def _all_shortest_paths(n, ef, et, w, s, t, d):
    """Every path s -> t of cost d[t], as tuples of edge ids (depth-first over tight edges)."""
    out = []

    def walk(v, suffix):
        if v == s and suffix:
            out.append(tuple(suffix))
            return
        for e in range(len(ef)):
            if et[e] == v and d[ef[e]] + w[e] == d[v] and et[e] != s:
                walk(ef[e], [e] + suffix)
    walk(t, [])
    return out


@pytest.mark.parametrize("seed", range(6))
def test_trees_against_bellman_ford_and_brute_force_tie_break(seed):
    """Small random graphs with weights in {1, 2}: many equal-cost paths, parallel edges."""
    rng = np.random.default_rng(seed)
    n, E = 6, 26
    ef = rng.integers(0, n, E); et = rng.integers(0, n, E)
    keep = ef != et
    ef, et = ef[keep], et[keep]
    w = rng.integers(1, 3, len(ef))
    src = np.arange(n)
    dist, pred = R.shortest_path_trees(n, ef, et, w, src)
    ties = 0
    for s in range(n):
        d = _bellman_ford(n, ef.tolist(), et.tolist(), w.tolist(), s)
        assert [float(x) for x in d] == dist[s].tolist()
        for t in range(n):
            if t == s or d[t] == float("inf"):
                assert pred[s, t] == -1
                continue
            paths = _all_shortest_paths(n, ef.tolist(), et.tolist(), w.tolist(), s, t, d)
            assert paths
            ties += len(paths) > 1
            # R38: walking back from t, always the smallest edge id among the tight inbound edges,
            # i.e. the path whose REVERSED edge sequence is lexicographically smallest
            want = min(paths, key=lambda p: p[::-1])
            got, v = [], t
            while v != s:
                got.append(int(pred[s, v])); v = int(ef[pred[s, v]])
            assert tuple(got[::-1]) == want
    assert ties > 0


def test_distances_against_floyd_warshall_on_config2():
    b = W.config2(n_vehicles=50)
    w = W.free_flow_weights(b)
    src = np.array([0, 17, 500, 1023])
    dist, _ = R.shortest_path_trees(b["n_nodes"], b["edge_from"], b["edge_to"], w, src)
    g = sp.csr_matrix((w.astype(np.float64), (b["edge_from"], b["edge_to"])), shape=(b["n_nodes"],) * 2)
    fw = floyd_warshall(g, directed=True)
    assert np.array_equal(dist, fw[src])


def test_rerouted_demand_has_the_properties_it_must_have(cfg1):
    b = cfg1
    o = Oracle(b)
    o.step(b["steps"])
    es = o.read_edge_stats()
    wf = W.free_flow_weights(b)
    mask = W.reroute_mask(b["n_vehicles"], 2)
    assert 0.4 < mask.mean() < 0.6
    off, edges, w = R.reroute(b, es["exited"], es["exit_steps_sum"], wf, mask)
    ef, et = b["edge_from"].astype(int), b["edge_to"].astype(int)
    old_off, old = b["route_off"].astype(int), b["route_edges"].astype(int)
    off = off.astype(int); edges = edges.astype(int)
    changed = 0
    for i in range(b["n_vehicles"]):
        new_r, old_r = edges[off[i]:off[i + 1]], old[old_off[i]:old_off[i + 1]]
        if not mask[i]:
            assert np.array_equal(new_r, old_r)
            continue
        assert ef[new_r[0]] == ef[old_r[0]] and et[new_r[-1]] == et[old_r[-1]]       # same origin, destination
        assert (et[new_r[:-1]] == ef[new_r[1:]]).all()                                 # contiguous
        assert w[new_r].sum() <= w[old_r].sum()                                        # never worse under w
        changed += not np.array_equal(new_r, old_r)
    assert changed > 0
    # and the new demand runs
    b2 = dict(b, route_off=off.astype(np.uint64), route_edges=edges.astype(np.uint32))
    o2 = Oracle(b2)
    o2.step(b["steps"], check=1)
    assert o2.read_counts()["n_arrived"] == b["n_vehicles"]


def test_measured_weights_pull_routes_off_a_congested_edge():
    """Two parallel one-lane roads A (short) and B (longer) between the same nodes; the first vehicle
    crawls (v0_mult 0.15) and nobody can pass it on A: the first run sends everybody down A behind
    it; with the measured weights the re-routed half moves to B ("reflects a behavioral adaptation by vehicles adapting to congestion")."""
    #   0 --e0--> 1 ==(e1 short 1 lane | e2 long 1 lane)==> 2 --e3--> 3
    ef = np.array([0, 1, 1, 2]); et = np.array([1, 2, 2, 3])
    length = np.array([200, 400, 520, 200]); lanes = np.array([2, 1, 1, 2])
    V = 300
    b = W.make_bundle("two_roads", 4, ef, et, length, lanes, np.full(4, 13.0), np.zeros(4), np.arange(V + 1) * 3,
                      np.tile([0, 1, 3], V), np.arange(V) * 0.7, 2400, v0_mult=np.r_[0.15, np.ones(V - 1)])
    o = Oracle(b)
    o.step(2400)
    es = o.read_edge_stats()
    w_free = W.free_flow_weights(b)
    assert w_free[1] < w_free[2]
    w = R.edge_weights(es["exited"], es["exit_steps_sum"], w_free)
    assert w[1] > w[2]                     # the short road measured slower than the empty long one
    mask = W.reroute_mask(V, 2)
    off, edges, _ = R.reroute(b, es["exited"], es["exit_steps_sum"], w_free, mask)
    second = edges[off[:-1].astype(int) + 1]
    assert (second[mask == 1] == 2).all() and (second[mask == 0] == 1).all()
