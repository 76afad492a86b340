"""Parity of ts_reroute against oracle/reroute.py: the
integer weights, every route (offsets and edges) and the simulation that follows on the new demand,
over the paper's four iterations (all / all / half / a quarter of the vehicles re-routed)."""
import numpy as np
import pytest

from paper_1807_01148_b200 import workload as W

pytestmark = pytest.mark.gpu


def _loop(bundle, iterations, steps=None, check_run=True, threads=1):
    import paper_1807_01148_b200 as pkg
    from oracle import Oracle
    from oracle import reroute as R
    steps = steps or bundle["steps"]
    cap = int(len(bundle["route_edges"]) * 2 + 1024)
    b = dict(bundle, params=dict(bundle["params"], route_capacity=cap))
    sim = pkg.Sim(b, "cuda:0")
    wf = W.free_flow_weights(b)
    changed_total = 0
    for it in range(iterations):
        orc = Oracle(b)
        orc.set_threads(threads)
        want = orc.step(steps, digests=True) if check_run else None
        if check_run:
            got = sim.step_digest(steps)
            bad = np.nonzero(want != got)[0]
            assert bad.size == 0, f"iteration {it}: first digest mismatch at step {int(bad[0]) + 1}"
        else:
            orc.step(steps); sim.step(steps)
        es = orc.read_edge_stats()
        gs = sim.read_edge_stats()
        for key in ("exited", "exit_steps_sum"):
            assert np.array_equal(es[key], gs[key]), key
        mask = W.reroute_mask(b["n_vehicles"], it)
        off, edges, w = R.reroute(b, es["exited"], es["exit_steps_sum"], wf, mask)
        info = sim.reroute(wf, mask)
        assert np.array_equal(info["w"], w), f"iteration {it}: weights"
        g_off, g_edges = sim.read_routes()
        assert np.array_equal(g_off, off), f"iteration {it}: route offsets"
        assert np.array_equal(g_edges, edges), f"iteration {it}: route edges"
        assert info["n_rerouted"] == int(mask.sum()) and info["route_entries"] == len(edges)
        changed_total += int((off != b["route_off"]).any() or not np.array_equal(edges, b["route_edges"]))
        b = dict(b, route_off=off, route_edges=edges)
        st = sim.read_counts()
        assert st["step"] == 0 and st["n_pending"] == b["n_vehicles"]       # ts_reroute resets
    # and the simulation on the last demand still matches
    if check_run:
        want = Oracle(b).step(min(steps, 1500), digests=True)
        assert np.array_equal(sim.step_digest(min(steps, 1500)), want)
    sim.close()
    return changed_total


def test_four_iterations_on_config1(cfg1):
    assert _loop(cfg1, 4) >= 3


def test_four_iterations_on_config2():
    assert _loop(W.config2(), 4, steps=6000) >= 3


def test_one_iteration_on_a_config3_subset():
    """cfg3_small: config 3's generator at 64x64 nodes, 50 000 vehicles from 512 origin nodes."""
    assert _loop(W.by_name("cfg3_small"), 2, steps=3600, threads=4) >= 1


def test_stop_and_trucks_with_rerouting(cfg1):
    assert _loop(W.with_trucks(W.with_controls(cfg1), share=0.2), 2) >= 1


def test_errors(cfg1):
    import paper_1807_01148_b200 as pkg
    sim = pkg.Sim(cfg1, "cuda:0")                         # route_capacity 0
    with pytest.raises(pkg.TsError) as e:
        sim.reroute(W.free_flow_weights(cfg1))
    assert e.value.code == pkg.binding.TS_EINVAL
    off, edges = sim.read_routes()                        # reading the routes works all the same
    assert np.array_equal(off, cfg1["route_off"]) and np.array_equal(edges, cfg1["route_edges"])
    sim.close()
    tight = dict(cfg1, params=dict(cfg1["params"], route_capacity=len(cfg1["route_edges"])))
    sim = pkg.Sim(tight, "cuda:0")
    sim.step(3600)
    wf = W.free_flow_weights(cfg1).copy()
    wf[:] = 1 << 20
    wf[::7] = 1                                           # detours: longer routes than the table holds
    try:
        sim.reroute(wf)
    except pkg.TsError as err:
        assert err.code == pkg.binding.TS_ENOMEM
        off, edges = sim.read_routes()
        assert np.array_equal(edges, cfg1["route_edges"])  # the routes in use are unchanged
    bad = wf.copy(); bad[3] = 0
    with pytest.raises(pkg.TsError):
        sim.reroute(bad)
    sim.close()
