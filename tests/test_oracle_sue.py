"""Pins of the static-assignment oracle (oracle/sue.py; PAPER.md:307-338 Frank-Wolfe, Eq. 3 BPR,
Eq. 6) against closed forms and the properties that define a user equilibrium."""
import numpy as np
import pytest
from scipy.optimize import brentq

from oracle import sue as S
from paper_1807_01148_b200 import workload as W


def test_bpr_and_its_integral_by_hand():
    """Eq. 3 with alpha = 0.15, beta = 4: at v = c the time is 1.15 t0; at v = 2c it is 3.4 t0.
    Eq. 6's integrand integrates to t0 (x + 0.15 x^5 / (5 c^4))."""
    t0, c = np.array([10.0]), np.array([100.0])
    assert S.bpr_time(t0, c, np.array([0.0]))[0] == 10.0
    assert S.bpr_time(t0, c, np.array([100.0]))[0] == pytest.approx(11.5)
    assert S.bpr_time(t0, c, np.array([200.0]))[0] == pytest.approx(34.0)
    assert S.objective(t0, c, np.array([100.0])) == pytest.approx(10.0 * (100 + 0.15 * 100 / 5))
    # derivative of the objective is the time
    x, h = 137.0, 1e-4
    num = (S.objective(t0, c, np.array([x + h])) - S.objective(t0, c, np.array([x - h]))) / (2 * h)
    assert num == pytest.approx(S.bpr_time(t0, c, np.array([x]))[0], rel=1e-8)


def test_two_parallel_roads_reach_the_closed_form_equilibrium():
    """Wardrop: with both roads used their times are equal.  Two roads between the same
    nodes, t0 = 10 / 15, c = 40 / 60, demand 100: the split solves t1(x) = t2(100 - x) -- a scalar
    equation solved here by Brent's method -- and Frank-Wolfe must converge to it."""
    ef, et = np.array([0, 0]), np.array([1, 1])
    t0, cap = np.array([10.0, 15.0]), np.array([40.0, 60.0])
    T = 100
    t1 = lambda x: 10.0 * (1 + 0.15 * (x / 40.0) ** 4)
    t2 = lambda x: 15.0 * (1 + 0.15 * (x / 60.0) ** 4)
    x_star = brentq(lambda x: t1(x) - t2(T - x), 0.0, T)
    x, t, hist = S.solve(2, ef, et, t0, cap, np.array([0]), np.array([1]), np.array([T]), iterations=30)
    assert x[0] == pytest.approx(x_star, abs=1e-3) and x[1] == pytest.approx(T - x_star, abs=1e-3)
    assert t[0] == pytest.approx(t[1], rel=1e-4)
    assert hist["step"][0] < 1.0 and all(0.0 <= a <= 1.0 for a in hist["step"])
    # low demand: everybody on the faster road, and the first step is the last
    x, t, hist = S.solve(2, ef, et, t0, cap, np.array([0]), np.array([1]), np.array([10]), iterations=3)
    assert x.tolist() == [10.0, 0.0] and t[0] < t[1]


def test_equilibrium_properties_on_a_grid():
    b = W.config2(n_vehicles=4000)
    inp = W.sue_inputs(b, horizon_s=120.0)        # heavy demand (v/c up to 2): congestion matters
    N, ef, et = b["n_nodes"], b["edge_from"], b["edge_to"]
    x, t, hist = S.solve(N, ef, et, inp["t0"], inp["cap"], inp["od_origin"], inp["od_dest"], inp["od_trips"], iterations=15)
    # step 3 of the algorithm: f never increases; it ends well below the all-or-nothing start
    f = np.array(hist["objective"])
    assert (np.diff(f) <= 1e-9 * f[0]).all() and f[-1] < 0.95 * f[0]
    # relative gap (x.t - y.t)/x.t -> 0 is Wardrop's condition: no flow on paths longer than the shortest
    assert hist["gap"][0] > 0.5 and hist["gap"][-1] < 0.05
    # conservation at every node: inflow - outflow = trips ending - trips starting there
    net = np.zeros(N)
    np.add.at(net, et, x); np.add.at(net, ef, -x)
    want = np.zeros(N)
    np.add.at(want, inp["od_dest"].astype(int), inp["od_trips"]); np.add.at(want, inp["od_origin"].astype(int), -inp["od_trips"].astype(float))
    assert np.allclose(net, want, atol=1e-6 * inp["od_trips"].sum())
    assert (x >= 0).all()


def test_all_or_nothing_loads_the_shortest_paths():
    b = W.config1()
    inp = W.sue_inputs(b)
    w = S.weights(inp["t0"], 1000.0)
    y = S.all_or_nothing(b["n_nodes"], b["edge_from"], b["edge_to"], w, inp["od_origin"], inp["od_dest"], inp["od_trips"])
    # total vehicle-weight loaded = sum over OD pairs of trips * shortest distance (Floyd-Warshall)
    import scipy.sparse as sp
    from scipy.sparse.csgraph import floyd_warshall
    g = sp.csr_matrix((w.astype(float), (b["edge_from"], b["edge_to"])), shape=(b["n_nodes"],) * 2)
    d = floyd_warshall(g, directed=True)
    want = sum(int(t) * d[int(o), int(dd)] for o, dd, t in zip(inp["od_origin"], inp["od_dest"], inp["od_trips"]))
    assert float((y.astype(float) * w).sum()) == want
    assert int(y.sum()) > 0
