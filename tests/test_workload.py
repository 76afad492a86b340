"""The seeded input generators (no GPU): shapes, contiguous shortest routes, determinism."""
import numpy as np
import scipy.sparse as sp
from scipy.sparse.csgraph import dijkstra

from paper_1807_01148_b200 import workload as W


def _check_bundle(b):
    ro, re = b["route_off"].astype(np.int64), b["route_edges"]
    assert ro[0] == 0 and (np.diff(ro) >= 1).all() and ro[-1] == len(re)
    inner = np.ones(len(re), bool); inner[ro[1:-1]] = False; inner[0] = False
    idx = np.nonzero(inner)[0]
    assert (b["edge_to"][re[idx - 1]] == b["edge_from"][re[idx]]).all()
    assert b["edge_len_m"].min() >= 40 and b["edge_lanes"].min() >= 1 and b["edge_lanes"].max() <= 8
    assert (b["depart_time_s"] >= 0).all()


def test_config1_shape_and_determinism():
    a, b = W.config1(), W.config1()
    assert W.bundle_sha256(a) == W.bundle_sha256(b)
    assert a["n_nodes"] == 16 and a["n_edges"] == 48 and a["n_vehicles"] == 500 and a["steps"] == 3600
    assert (a["edge_len_m"] == 200).all() and (a["edge_lanes"] == 2).all() and (a["edge_vlim"] == 15).all()
    assert (a["node_ctrl"] == W.CTRL_PRIORITY).all() and a["depart_time_s"].max() <= 300
    _check_bundle(a)


def test_routes_are_shortest_paths():
    b = W.config2(n_vehicles=400, grid=8, steps=10, workers=1)
    _check_bundle(b)
    w = b["edge_len_m"] / b["edge_vlim"].astype(np.float64)
    g = sp.csr_matrix((w, (b["edge_from"], b["edge_to"])), shape=(b["n_nodes"],) * 2)
    ro = b["route_off"].astype(np.int64)
    o = b["edge_from"][b["route_edges"][ro[:-1]]]
    d = b["edge_to"][b["route_edges"][ro[1:] - 1]]
    dist = dijkstra(g, indices=np.unique(o))
    row = np.searchsorted(np.unique(o), o)
    cost = np.add.reduceat(w[b["route_edges"]], ro[:-1])
    assert np.allclose(cost, dist[row, d], rtol=1e-9)


def test_parallel_routing_equals_serial():
    a = W.config2(n_vehicles=600, grid=10, steps=10, workers=1)
    b = W.config2(n_vehicles=600, grid=10, steps=10, workers=3)
    assert W.bundle_sha256(a) == W.bundle_sha256(b)


def test_config3_and_5_small():
    b = W.config3(n_vehicles=3000, grid=24, steps=100, n_origin_nodes=64, workers=2)
    _check_bundle(b)
    assert set(np.unique(b["edge_lanes"])) <= {1, 2, 4} and (b["edge_vlim"][b["edge_lanes"] == 4] == 29).all()
    assert set(np.unique(b["node_ctrl"])) <= {W.CTRL_PRIORITY, W.CTRL_SIGNAL}
    b5 = W.config5(n_vehicles=2000, grid=16, steps=100, core=4, workers=2)
    _check_bundle(b5)
    assert len(np.unique(b5["edge_from"][b5["route_edges"][b5["route_off"][:-1].astype(np.int64)]])) <= 16


def test_variant_helpers_keep_the_demand_and_only_add_inputs():
    """with_trucks / with_controls, the re-routing inputs (row 1) and the
    static-assignment inputs (row 5) are derived from a config without touching its network or routes."""
    b = W.config1()
    t = W.with_trucks(b, share=0.3)
    assert t["veh_type"].dtype == np.uint8 and 0.2 < t["veh_type"].mean() < 0.4
    assert t["params"]["n_types"] == 2 and np.array_equal(t["route_edges"], b["route_edges"])
    assert W.bundle_sha256(t) != W.bundle_sha256(b)
    c = W.with_controls(b, amber_steps=4)
    assert (c["node_ctrl"] == W.CTRL_STOP).all() and c["params"]["amber_steps"] == 4
    c2 = W.with_controls(W.config2(n_vehicles=10))
    assert set(np.unique(c2["node_ctrl"])) == {W.CTRL_SIGNAL, W.CTRL_SIGNAL_NM}
    wf = W.free_flow_weights(b)
    assert wf.dtype == np.uint32 and (wf >= 1).all() and (wf <= 1 << 20).all()
    # 200 m at 15 m/s on 2 lanes: 200 / (15 sqrt 2) s = 18.86 steps of 0.5 s = 4827 units of 1/256 step
    assert wf[0] == round(200 / (15 * 2 ** 0.5) / 0.5 * 256)
    shares = [W.reroute_mask(100000, it).mean() for it in range(4)]
    assert shares[0] == shares[1] == 1.0 and abs(shares[2] - 0.5) < 0.01 and abs(shares[3] - 0.25) < 0.01
    assert np.array_equal(W.reroute_mask(1000, 2), W.reroute_mask(1000, 2))             # seeded
    s = W.sue_inputs(b, horizon_s=60.0)
    assert int(s["od_trips"].sum()) == b["n_vehicles"] and (s["od_origin"] != s["od_dest"]).all()
    assert np.allclose(s["t0"], 200 / 15.0) and np.allclose(s["cap"], 900.0 * 2 / 3600.0 * 60.0)
