"""Parity of ts_sue_solve (PAPER.md:307-338 Frank-Wolfe + BPR) against
oracle/sue.py.  The all-or-nothing flows are integers on both sides (bit-exact: same trees, same
tie-break); the line search sums fp64 terms in a different order, so steps, flows and objective are
compared within a tolerance derived from that: |sum error| <= E * 2^-53 relative, bisection to 2^-40,
flows are convex combinations of integers <= total trips -> relative 1e-9."""
import numpy as np
import pytest

from paper_1807_01148_b200 import workload as W

pytestmark = pytest.mark.gpu


def _check(n_nodes, ef, et, inp, iterations, rtol=1e-9):
    import paper_1807_01148_b200 as pkg
    from oracle import sue as S
    args = (n_nodes, ef, et, inp["t0"], inp["cap"], inp["od_origin"], inp["od_dest"], inp["od_trips"])
    x, t, hist = S.solve(*args, iterations=iterations)
    gx, gt, info = pkg.sue_solve(*args, iterations=iterations)
    scale = float(np.sum(inp["od_trips"]))
    assert np.allclose(info["step"], hist["step"], rtol=0, atol=1e-9)
    assert np.allclose(gx, x, rtol=0, atol=rtol * scale)
    assert np.allclose(gt, t, rtol=1e-8)
    assert np.allclose(info["objective"], hist["objective"], rtol=1e-10)
    assert np.allclose(info["gap"], hist["gap"], rtol=1e-7, atol=1e-10)
    return info


def test_two_roads_closed_form():
    ef, et = np.array([0, 0]), np.array([1, 1])
    inp = dict(t0=np.array([10.0, 15.0]), cap=np.array([40.0, 60.0]), od_origin=np.array([0]), od_dest=np.array([1]),
               od_trips=np.array([100]))
    import paper_1807_01148_b200 as pkg
    from scipy.optimize import brentq
    _check(2, ef, et, inp, 30)
    x, t, info = pkg.sue_solve(2, ef, et, inp["t0"], inp["cap"], inp["od_origin"], inp["od_dest"], inp["od_trips"], iterations=30)
    x_star = brentq(lambda a: 10.0 * (1 + 0.15 * (a / 40.0) ** 4) - 15.0 * (1 + 0.15 * ((100 - a) / 60.0) ** 4), 0.0, 100.0)
    assert x[0] == pytest.approx(x_star, abs=1e-3) and t[0] == pytest.approx(t[1], rel=1e-4)


def test_config1_and_config2_demand():
    b = W.config1()
    _check(b["n_nodes"], b["edge_from"], b["edge_to"], W.sue_inputs(b, horizon_s=60.0), 20)
    b = W.config2(n_vehicles=4000)
    info = _check(b["n_nodes"], b["edge_from"], b["edge_to"], W.sue_inputs(b, horizon_s=120.0), 15)
    assert info["gap"][0] > 0.5 and info["gap"][-1] < 0.05
    assert (np.diff(info["objective"]) <= 1e-9 * info["objective"][0]).all()


def test_sue_errors():
    import paper_1807_01148_b200 as pkg
    ef, et = np.array([0, 0]), np.array([1, 1])
    with pytest.raises(pkg.TsError):
        pkg.sue_solve(2, ef, et, np.array([10.0, 0.0]), np.array([40.0, 60.0]), [0], [1], [5])
    with pytest.raises(pkg.TsError):
        pkg.sue_solve(2, ef, np.array([1, 7]), np.array([10.0, 1.0]), np.array([40.0, 60.0]), [0], [1], [5])
