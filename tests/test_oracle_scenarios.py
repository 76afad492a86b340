"""Scenario pins for the rules SURVEY.md lists as pinned oracle<->GPU only: the discretionary
lane-change incentive (MOBIL, reading R10), hold-at-line after a lost claim (R15) and departure
ordering (R18/R19).  Each scenario is small enough to re-derive the expected behaviour here, in
Python and fp64, from the rule as DESIGN.md section 2 states it -- not from the oracle's code."""
import math

import numpy as np

from oracle import Oracle
from paper_1807_01148_b200 import workload as W
from test_oracle_pins import corridor

P = W.DEFAULT_PARAMS


def _idm64(v, v0, s=None, dv=0.0):
    free = 1.0 - (v / v0) ** 4
    if s is None:
        return P["a"] * free
    sstar = P["s0"] + max(0.0, v * P["T"] + v * dv / (2.0 * math.sqrt(P["a"] * P["b"])))
    return P["a"] * (free - (sstar / max(s, 0.5)) ** 2)


def test_mobil_overtake_happens_exactly_when_the_incentive_passes_the_threshold():
    """Two lanes, a slow leader (id 0) and a faster follower (id 1) behind it in lane 0, lane 1
    empty.  With no vehicle in the target lane the rule reduces to
        a(1 - (v/v0)^4)  -  idm(v, v0, s, dv)  >  lc_threshold,
    evaluated only on the follower's turns (even k for a move to the left lane, ((k>>1)+id) % 4 == 0,
    x >= entry zone, not able to leave the edge).  The follower must change lane at the FIRST turn
    on which that holds and at none before."""
    v0 = 15.0
    rejected_turns = accepted_turns = 0
    for headway_s in (6.0, 14.0, 25.0, 31.0):        # how far behind the follower starts
        b = corridor(length=20000, lanes=2, vlim=v0, departs=(0.0, headway_s), v0_mult=np.array([0.5, 1.0]), steps=900)
        o = Oracle(b)
        changed_at = None
        for k in range(900):
            st = o.read_state()
            o.step(1, check=1)
            after = o.read_state()
            if st["status"][1] != 1 or st["lane"][1] != 0:
                continue
            x, v = float(st["x"][1]), float(st["v"][1])
            turn = (k % 2 == 0) and ((k >> 1) + 1) % P["lc_period"] == 0 and x >= P["entry_zone_cells"]
            gap = float(st["cell"][0]) - P["veh_len"] - x                 # perceived: leader's cell index
            v_lead = round(float(st["v"][0]) * 4.0) / 4.0                  # perceived: 0.25 m/s grid
            near = st["lane"][0] == 0 and 0 < st["cell"][0] - st["cell"][1] <= P["lookahead_cells"]
            a_c = _idm64(v, v0, gap, v - v_lead) if near else _idm64(v, v0)
            inc = _idm64(v, v0) - a_c
            if abs(inc - P["lc_threshold"]) < 1e-3:
                continue                                                   # too close to call in fp64 vs fp32
            want = turn and inc > P["lc_threshold"]
            got = after["lane"][1] == 1
            assert got == want, (headway_s, k, inc, turn)
            if turn:
                rejected_turns += not got
                accepted_turns += got
            if got:
                changed_at = k
                break
        assert changed_at is not None
        # and it then passes the slow leader, who stays where it is
        o.step(600)
        st = o.read_state()
        assert st["x"][1] > st["x"][0] and st["lane"][0] == 0
    assert rejected_turns >= 4 and accepted_turns == 4


def test_mobil_no_change_without_incentive_and_none_into_an_unsafe_gap():
    # equal desired speeds, generous spacing: the incentive never reaches the threshold
    b = corridor(length=20000, lanes=2, departs=(0.0, 20.0, 40.0), steps=600)
    o = Oracle(b)
    o.step(600, check=1)
    assert o.counters()["lc_accepts"] == 0 and o.counters()["lc_evals"] > 0
    assert (o.read_state()["lane"] == 0).all()
    # dense platoon behind a crawler: changes happen, and gap acceptance keeps every lag gap >= s0
    # at the moment of the change (I2/I3 are asserted every step by check=1; P4 by check=2)
    V = 40
    b = corridor(length=6000, lanes=2, departs=np.arange(V) * 2.0, v0_mult=np.r_[0.2, np.ones(V - 1)], steps=900)
    o = Oracle(b)
    prev = o.read_state()
    seen = 0
    for _ in range(900):
        o.step(1, check=2)
        st = o.read_state()
        moved = np.nonzero((st["status"] == 1) & (prev["status"] == 1) & (st["lane"] != prev["lane"]))[0]
        for i in moved:
            same = (prev["status"] == 1) & (prev["lane"] == st["lane"][i]) & (np.arange(V) != i)
            behind = same & (prev["cell"] < prev["cell"][i])
            if behind.any():
                lag = prev["cell"][behind].max()
                assert float(prev["x"][i]) - P["veh_len"] - (lag + 1) >= P["s0"]
            ahead = same & (prev["cell"] >= prev["cell"][i])
            if ahead.any():
                assert prev["cell"][ahead].min() - P["veh_len"] - float(prev["x"][i]) >= P["s0"]
            seen += 1
        prev = st
    assert seen >= 5


def test_loser_of_a_claim_is_held_at_the_line_and_the_lowest_id_goes_first():
    """R15: two vehicles reach a PRIORITY node in the same step from different edges.  The lower
    id crosses; the other one stands at C - 1/16 with v = 0 after that step and crosses later."""
    ef, et = np.array([0, 1, 2]), np.array([2, 2, 3])            # A->X, B->X, X->C
    V = 2
    route_off = np.array([0, 2, 4])
    route_edges = np.array([1, 2, 0, 2])                          # id 0 comes from B, id 1 from A
    b = W.make_bundle("tie", 4, ef, et, np.full(3, 120), np.full(3, 1), np.full(3, 15.0),
                      np.array([0, 0, W.CTRL_PRIORITY, 0]), route_off, route_edges, np.zeros(V), 300)
    o = Oracle(b)
    held = False
    for k in range(300):
        before = o.read_state()
        o.step(1, check=2)
        st = o.read_state()
        if before["edge"][0] == 1 and st["edge"][0] == 2:         # id 0 crossed in this step
            # symmetric approach: id 1 tried in the same step, lost, and is held
            assert st["edge"][1] == 0 and st["x"][1] == np.float32(120 - 0.0625) and st["v"][1] == 0.0
            held = True
        if held and st["edge"][1] == 2:
            break
    assert held and o.counters()["cross_lost"] >= 1
    o.step(200)
    assert o.read_state()["n_arrived"] == 2


def test_departures_are_fifo_by_step_then_id_and_wait_for_a_clear_entry():
    """R18/R19: vehicles of one origin edge enter in (ceil(t/dt), id) order, never two in one step,
    each at x = 0, v = 0 in lane 0, and only when cells [0, 7) of lane 0 are free."""
    t = np.array([3.2, 0.0, 3.2, 0.4, 0.0, 10.0, 0.26])
    b = corridor(length=3000, lanes=2, departs=t, steps=200)
    o = Oracle(b)
    o.step(200, check=1)
    st = o.read_state()
    dep_step = np.ceil(t.astype(np.float32).astype(np.float64) / P["dt"])
    order = np.lexsort((np.arange(len(t)), dep_step))
    ins = st["insert_step"][order].astype(int)
    assert (np.diff(ins) > 0).all()                               # FIFO, one per step at most
    assert (st["insert_step"] >= dep_step + 1).all()              # never early
    assert ins[0] == int(dep_step[order[0]]) + 1                  # the first one is on time
    # a successor waits until its predecessor's front bumper has left cells [0, 7): from rest that
    # takes several steps, so consecutive entries are > 1 step apart while the queue is backed up
    backed_up = dep_step[order][1:] + 1 < ins[1:]
    assert backed_up.any() and (np.diff(ins)[backed_up] >= 5).all()


def test_utilisation_of_a_jammed_edge_is_one():
    """PAPER.md:446 defines utilisation against the number of vehicles that fit, length x lanes /
    (vehicle length + lead gap).  A one-lane edge behind a permanently red light fills up with a
    standing queue at veh_len + s0 = 7 m spacing (pin P3), so its sampled utilisation must come out
    at 1 (+- one vehicle), and its sampled speed at 0; the empty edge beyond the light at 0."""
    from oracle import utilisation
    N = 3
    sig = (np.full(N, 1), np.full(N, 1_000_000), np.full(N, 1))
    b = corridor(n_edges=2, length=210, departs=np.arange(60) * 3.0, ctrl=W.CTRL_SIGNAL, sig=sig, steps=3000)
    o = Oracle(b)
    o.step(2400)                      # the queue has filled the edge
    o.read_edge_stats(reset=True)
    o.step(600)                       # five samples of the standing queue
    es = o.read_edge_stats()
    util, speed = utilisation(es, b)
    assert es["n_samples"] == 5
    assert abs(util[0] - 1.0) <= 7.0 / 210 + 1e-9 and util[1] == 0.0
    assert speed[0] < 0.05
    # by hand: 14 vehicle-samples over 2 samples on 100 m x 2 lanes -> 7 / (200 / 7)
    es2 = dict(sample_count_sum=np.array([14]), sample_speedcode_sum=np.array([14 * 40]), n_samples=2)
    u2, v2 = utilisation(es2, dict(b, edge_len_m=np.array([100]), edge_lanes=np.array([2])))
    assert u2[0] == 7.0 / (200.0 / 7.0) and v2[0] == 10.0
