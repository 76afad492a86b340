"""Invariants I1-I8, brute force P4 and degenerate cases P5 of the oracle (no GPU).

orc_step(check=1) asserts, after every step: I1 conservation (counts, entered-exited,
on-route), I2 exclusivity and I3 order (per-lane lists strictly increasing in cell), I4
speed range, I5 position range and per-step advance bound, I7 arbitration (<= 1 entry per
lane, <= 1 crossing per PRIORITY node, nobody crosses on red).  check=2 adds P4: every
neighbour the lane lists return is re-derived by an O(V^2) search over raw (edge, lane, x).
"""
import numpy as np
import pytest

from oracle import Oracle, OracleError
from paper_1807_01148_b200 import workload as W
from test_oracle_pins import corridor


def small_signal_grid(seed=7, n_vehicles=1500, grid=6, steps=1500, lanes=(1, 2, 3)):
    """A small cousin of config 2 that exercises signals, 1-3 lanes and mandatory changes."""
    rng = np.random.default_rng(seed)
    N = grid * grid
    und = W._grid_undirected(grid, grid)
    U = len(und)
    ulen = rng.integers(60, 300, U)
    ulanes = rng.choice(lanes, U)
    ulim = np.array([0.0, 13.0, 17.0, 22.0])[ulanes]
    ef, et, length, ln, vlim = W._directed(und, ulen, ulanes, ulim)
    ctrl = rng.choice([W.CTRL_FREE, W.CTRL_PRIORITY, W.CTRL_SIGNAL], N, p=[0.1, 0.3, 0.6])
    sig = W._signal_arrays(rng, N, et, ctrl == W.CTRL_SIGNAL, 20, 4)
    origins = rng.integers(0, N, n_vehicles)
    dests = (origins + rng.integers(1, N, n_vehicles)) % N
    depart = rng.random(n_vehicles) * 200.0
    xy = np.stack([np.arange(N) % grid, np.arange(N) // grid], 1) * 200.0
    return W._finish("small_signal_grid", rng, N, ef, et, length, ln, vlim, ctrl, sig, origins,
                     dests, depart, steps, rng.uniform(0.9, 1.1, n_vehicles), None, xy, 1)


def test_cfg1_all_checks_and_completion(cfg1):
    """Config 1 in full with I1-I7 and P4 every step; everybody arrives (no deadlock)."""
    o = Oracle(cfg1)
    o.step(cfg1["steps"], check=2)
    st = o.read_state()
    assert st["n_arrived"] == cfg1["n_vehicles"] and st["n_active"] == 0 and st["n_pending"] == 0
    es = o.read_edge_stats()
    assert es["entered"].sum() == es["exited"].sum() == len(cfg1["route_edges"])
    # time on edges adds up to each vehicle's trip time (I1, exit_steps_sum definition)
    assert es["exit_steps_sum"].sum() == (st["arrive_step"].astype(np.int64) - st["insert_step"]).sum()
    # departures never precede their time: insert_step >= ceil(t/dt) + 1
    dep = np.ceil(cfg1["depart_time_s"].astype(np.float64) / 0.5)
    assert (st["insert_step"] >= dep + 1).all()
    c = o.counters()
    assert c["lc_accepts"] > 0 and c["cross_lost"] > 0 and c["crossings"] + 500 == es["entered"].sum()


def test_mixed_controls_all_checks():
    b = small_signal_grid()
    o = Oracle(b)
    o.step(b["steps"], check=2)
    c = o.counters()
    # the scenario must actually exercise every branch it is meant to pin
    for key in ("lc_accepts", "lc_mandatory", "cross_lost", "held_red", "cap_bound", "crossings"):
        assert c[key] > 0, key


def test_i8_order_independence(cfg1):
    a = Oracle(cfg1).step(1200, digests=True)
    b = Oracle(cfg1).step(1200, digests=True, order_seed=12345)
    assert (a == b).all()
    b2 = small_signal_grid(n_vehicles=600, steps=600)
    assert (Oracle(b2).step(600, digests=True) == Oracle(b2).step(600, digests=True, order_seed=99)).all()


def test_threaded_intent_loop_changes_nothing():
    """orc_set_threads(n): the intent loop of step 2 on n host threads (used by make_golden.py for
    the multi-hour traces) gives the same digests, state, edge statistics, emission totals and
    work counters as the sequential program, with the invariant checks on."""
    b = small_signal_grid(n_vehicles=1200, steps=900)
    b = dict(b, params=dict(b["params"], emissions=1))
    one, many = Oracle(b), Oracle(b)
    many.set_threads(5)
    assert (one.step(900, digests=True, check=1) == many.step(900, digests=True, check=1)).all()
    assert one.counters() == many.counters()
    s1, s2 = one.read_state(), many.read_state()
    for k in s1:
        assert np.array_equal(s1[k], s2[k]), k
    e1, e2 = one.read_edge_stats(), many.read_edge_stats()
    for k in e1:
        assert np.array_equal(e1[k], e2[k]), k
    m1, m2 = one.read_emissions(), many.read_emissions()
    assert np.array_equal(m1["co_g"].view(np.uint32), m2["co_g"].view(np.uint32))
    assert np.array_equal(m1["fuel_ml"].view(np.uint32), m2["fuel_ml"].view(np.uint32))


def test_digest_sensitivity(cfg1):
    """The digest separates runs that differ in one parameter (it is not constant)."""
    b = dict(cfg1); b["params"] = dict(cfg1["params"], T=1.6)
    a = Oracle(cfg1).step(600, digests=True)
    c = Oracle(b).step(600, digests=True)
    assert (a != c).any() and len(set(a.tolist())) > 500


def test_sampling_counts(cfg1):
    """one sample per minute (120 steps); counts equal the active vehicles then."""
    o = Oracle(cfg1)
    total = 0
    code_total = 0
    for _ in range(10):
        o.step(120)
        st = o.read_state()
        act = st["status"] == 1
        total += int(act.sum())
        code_total += int(np.minimum(254, (st["v"][act] * np.float32(4.0) + np.float32(0.5)).astype(np.int64)).sum())
    es = o.read_edge_stats()
    assert es["n_samples"] == 10
    assert es["sample_count_sum"].sum() == total and total > 0
    assert es["sample_speedcode_sum"].sum() == code_total
    es2 = o.read_edge_stats(reset=True)
    assert o.read_edge_stats()["sample_count_sum"].sum() == 0 and es2["n_samples"] == 10


# ------------------------------------------------------------------ P5 degenerate cases

def test_p5_no_lane_changes_when_disabled(cfg1):
    b = dict(cfg1); b["params"] = dict(cfg1["params"], lc_period=0)
    o = Oracle(b)
    for _ in range(30):
        o.step(40, check=1)
        st = o.read_state()
        assert (st["lane"][st["status"] == 1] == 0).all()     # inserted in lane 0, index preserved
    assert o.counters()["lc_evals"] == 0


def test_p5_always_green_equals_free():
    """A SIGNAL node with one inbound edge and no all-red is always green: same run as FREE."""
    dep = np.arange(8) * 3.0
    free = corridor(n_edges=3, length=300, lanes=2, departs=dep, ctrl=W.CTRL_FREE)
    sig = corridor(n_edges=3, length=300, lanes=2, departs=dep, ctrl=W.CTRL_SIGNAL,
                   sig=(np.full(4, 5), np.zeros(4), np.full(4, 3)))
    assert (Oracle(free).step(400, digests=True, check=1) == Oracle(sig).step(400, digests=True, check=1)).all()


def test_p5_priority_without_conflict_equals_free():
    dep = np.arange(8) * 3.0
    free = corridor(n_edges=3, length=300, departs=dep, ctrl=W.CTRL_FREE)
    prio = corridor(n_edges=3, length=300, departs=dep, ctrl=W.CTRL_PRIORITY)
    assert (Oracle(free).step(400, digests=True) == Oracle(prio).step(400, digests=True)).all()


def test_priority_node_one_at_a_time():
    """PAPER.md:402 'allows just one vehicle at a time into the intersection': two streams
    meeting at a PRIORITY node never cross it in the same step, and the lower id goes first."""
    # edges: 0: A->X, 1: B->X, 2: X->C (2 lanes so lane claims alone would not serialise), 3: X->D
    ef, et = np.array([0, 1, 2, 2]), np.array([2, 2, 3, 4])
    V = 40
    first = np.arange(V) % 2
    route_off = np.arange(V + 1) * 2
    route_edges = np.stack([first, 2 + first], 1).ravel()
    b = W.make_bundle("merge", 5, ef, et, np.full(4, 150), np.full(4, 1), np.full(4, 15.0),
                      np.array([0, 0, W.CTRL_PRIORITY, 0, 0]), route_off, route_edges,
                      (np.arange(V) // 2) * 4.0, 600)
    o = Oracle(b)
    prev = o.read_edge_stats()
    both = 0
    for _ in range(600):
        o.step(1, check=2)
        es = o.read_edge_stats()
        crossed = int(es["entered"][2] - prev["entered"][2]) + int(es["entered"][3] - prev["entered"][3])
        assert crossed <= 1
        prev = es
    assert o.counters()["cross_lost"] > 0           # the conflict did occur
    assert o.read_state()["n_arrived"] == V


def test_validation_rejects_bad_input(cfg1):
    bad = dict(cfg1); bad["edge_len_m"] = cfg1["edge_len_m"].copy(); bad["edge_len_m"][0] = 8
    with pytest.raises(OracleError):
        Oracle(bad)
    bad = dict(cfg1); bad["route_edges"] = cfg1["route_edges"].copy(); bad["route_edges"][1] = bad["route_edges"][0]
    with pytest.raises(OracleError):
        Oracle(bad)
    bad = dict(cfg1); bad["params"] = dict(cfg1["params"], lookahead_cells=100)
    with pytest.raises(OracleError):
        Oracle(bad)


def _closest_cells(bundle, steps):
    """Smallest difference between the cells (floor of x) of two vehicles of one lane over a run of the oracle."""
    o = Oracle(bundle)
    closest = 1 << 30
    for _ in range(steps):
        o.step(1, check=1)
        st = o.read_state()
        act = np.nonzero(st["status"] == 1)[0]
        if act.size < 2:
            continue
        cell = np.floor(st["x"][act]).astype(np.int64)
        key = st["edge"][act].astype(np.int64) * 16 + st["lane"][act]
        order = np.lexsort((cell, key))
        same = key[order][1:] == key[order][:-1]
        if same.any():
            closest = min(closest, int((cell[order][1:] - cell[order][:-1])[same].min()))
    return closest, o.counters()


def test_cells_of_one_lane_stay_a_vehicle_length_apart():
    """What lets the CUDA atlas keep ONE speed-code byte per 4 cells: under the rule
    set the cells of two vehicles of a lane differ by at least ceil(L) through following (E2 caps the advance
    at the gap to the leader's cell minus its length), by more than L - 1 after a lane change with a lag
    vehicle (G2), and entrants need insert_clear free cells -- so with L >= 4 m never less than 4.  Checked on
    the oracle at every step of dense platoons with forced merges, a signalised grid with queues, trucks, and
    a queue of 4 m vehicles standing 0.25 m apart."""
    from test_oracle_lane_change_referee import _platoon_scenario
    for politeness in (0.2, 0.5):
        closest, cnt = _closest_cells(_platoon_scenario(politeness, 5), 1400)
        assert cnt["lc_accepts"] > 100 and closest >= 5, (closest, cnt)
    closest, cnt = _closest_cells(small_signal_grid(), 1500)
    assert cnt["lc_accepts"] > 50 and closest >= 5, closest
    closest, _ = _closest_cells(W.with_trucks(small_signal_grid(n_vehicles=900, steps=700), share=0.3), 700)
    assert closest >= 5, closest
    g = small_signal_grid()
    tight = dict(g, params=dict(g["params"], veh_len=4.0, s0=0.25, insert_clear_cells=4))
    closest, cnt = _closest_cells(tight, 1500)
    assert 4 <= closest <= 5 and cnt["lc_accepts"] > 50, closest
