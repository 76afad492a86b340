"""Pins of the oracle's vehicle types (reading R31) and control variants
(readings R34 STOP with a persistent node owner, R35 one signal phase per movement,
R36 amber) against things other than the oracle: the closed forms of Eq. 7 with the truck's own
`a`, length and speed cap; explicit phase tables; the rule text applied to the recorded states."""
import math

import numpy as np
import pytest

from oracle import Oracle, lib
from paper_1807_01148_b200 import workload as W
from test_oracle_invariants import small_signal_grid
from test_oracle_lane_change_referee import Referee, _platoon_scenario
from test_oracle_pins import _rows, _t_closed, corridor

P = W.DEFAULT_PARAMS
TRUCK = W.TRUCK_PARAMS


# ------------------------------------------------------------------ vehicle types

def test_lone_truck_follows_the_closed_form_with_its_own_a_and_speed_cap():
    """P1 for a truck: Eq. 7's free term with a = type_a and v0 = min(limit, type_vmax)."""
    a_t, vmax = 0.5, 10.0
    prm = dict(n_types=2, type_len=(5, 12, 0, 0), type_a=(1.0, a_t, 0, 0), type_vmax=(1000.0, vmax, 0, 0))
    b = dict(corridor(length=30000, vlim=15.0, steps=400, params=prm), veh_type=np.array([1], np.uint8))
    o = Oracle(b)
    worst, v = 0.0, 0.0
    for k in range(1, 300):
        o.step(1, check=1)
        st = o.read_state()
        v = float(st["v"][0])
        t = (k - 1) * P["dt"]
        lo, hi = 0.0, 1.0 - 1e-12
        for _ in range(80):
            mid = 0.5 * (lo + hi)
            lo, hi = (mid, hi) if _t_closed(mid, vmax, a_t) < t else (lo, mid)
        worst = max(worst, abs(v - lo * vmax))
        assert v <= vmax
    assert worst <= 0.10 and v > 0.99 * vmax
    # the same vehicle as a car would be past 10 m/s long before
    car = Oracle(corridor(length=30000, vlim=15.0, steps=400))
    car.step(60)
    assert car.read_state()["v"][0] > 12.0


@pytest.mark.parametrize("leader_type,follower_type,follower_vmax", [(1, 0, 1000.0), (0, 1, 1000.0), (1, 1, 13.0)])
def test_p2_equilibrium_gap_uses_the_leaders_length_and_the_followers_cap(leader_type, follower_type, follower_vmax):
    """P2 (s_e = (s0 + vT)/sqrt(1 - (v/v0)^4), tests/golden/idm_equilibrium_gap.txt) with trucks:
    the gap the follower keeps is measured to the leader's REAR, i.e. with the leader's own length
    (12 m for a truck), whatever the follower's length or acceleration; a follower whose type caps
    its speed at 13 m/s has v0 = 13 in the formula."""
    v0e, v, s0, T, s_e_car = _rows("idm_equilibrium_gap.txt")[0]
    lens, accs = (5.0, 12.0), (1.0, 0.5)
    prm = dict(n_types=2, type_len=lens + (0, 0), type_a=accs + (0, 0), type_vmax=(1000.0, follower_vmax, 0, 0))
    b = corridor(length=40000, vlim=v0e, departs=(0.0, 12.0), v0_mult=np.array([v / v0e, 1.0]), params=prm)
    b = dict(b, veh_type=np.array([leader_type, follower_type], np.uint8))
    o = Oracle(b)
    o.step(3000, check=1)
    st = o.read_state()
    v0_f = min(v0e, follower_vmax if follower_type == 1 else 1000.0)
    s_e = (s0 + v * T) / math.sqrt(1 - (v / v0_f) ** 4)
    if v0_f == v0e:
        assert s_e == pytest.approx(s_e_car, abs=1e-3)
    perceived = float(st["cell"][0]) - lens[leader_type] - float(st["x"][1])
    assert st["v"][0] == pytest.approx(v, abs=1e-3) and st["v"][1] == pytest.approx(v, abs=0.01)
    # at v/v0 = 12/13 the equilibrium is stiff (ds_e/dv = 20 m per m/s) and x is ~4e4 m (fp32 ulp 4 mm)
    assert abs(perceived - s_e) <= (0.01 if v0_f == v0e else 0.03), (perceived, s_e)


def test_every_lane_change_decision_with_trucks_in_the_platoons():
    """The referee of test_oracle_lane_change_referee.py with 30 % trucks: gaps use the length of
    the vehicle AHEAD (leader, or the changer for the lag gap), G2/G3 and the follower terms use
    the lag vehicle's own `a` and capped limit."""
    b = _platoon_scenario(0.2, 5)
    rng = np.random.default_rng(3)
    b = dict(b, veh_type=(rng.random(b["n_vehicles"]) < 0.3).astype(np.uint8),
             params=dict(b["params"], n_types=2, type_len=(5.0, 12.0, 0, 0), type_a=(1.0, 0.5, 0, 0),
                         type_vmax=(1000.0, 14.0, 0, 0), insert_clear_cells=14))
    t = Referee(b).run(1400)
    assert t["turns"] > 3000 and t["accepted"] > 100 and t["skipped"] < 0.05 * t["turns"], t
    assert t["g2_kinematic_rejects"] >= 3 and t["g3_rejects"] >= 3 and t["polite_flips_to_no"] >= 3, t


def test_bodies_never_overlap_with_trucks():
    """I2 for bodies: on every lane the rear of the vehicle ahead (x - its length) stays ahead of
    the front of the one behind, trucks included, through signals, lane changes and queues."""
    b = W.with_trucks(small_signal_grid(n_vehicles=900, steps=700), share=0.3)
    lens = np.asarray(b["params"]["type_len"])[b["veh_type"]]
    o = Oracle(b)
    closest = 1e9
    for _ in range(700):
        o.step(1, check=1)
        st = o.read_state()
        act = np.nonzero(st["status"] == 1)[0]
        key = st["edge"][act].astype(np.int64) * 16 + st["lane"][act]
        order = act[np.lexsort((st["x"][act], key))]
        same = (st["edge"][order][1:] == st["edge"][order][:-1]) & (st["lane"][order][1:] == st["lane"][order][:-1])
        gap = (st["x"][order][1:] - lens[order][1:]) - st["x"][order][:-1]
        if same.any():
            closest = min(closest, float(gap[same].min()))
    assert closest > 0.0, closest
    assert o.counters()["lc_accepts"] > 0 and (b["veh_type"] == 1).sum() > 100


# ------------------------------------------------------------------ signals: amber, n*m phases

def test_signal_phase_function_against_an_explicit_timetable():
    """"the geometric combination nm of necessary traffic phasing ... round robin":
    the timetable written out step by step (phase (i, j) number i*m + j, `green` steps of green,
    `amber` of amber, `allred` of red, repeating), compared with orc_signal_phase at every step,
    for every movement; with n_out = 0 the same with one phase per inbound edge."""
    L = lib()
    green, amber, allred, off = 5, 2, 3, 4
    for n_in, n_out in ((3, 2), (2, 0), (4, 3), (1, 1)):
        phases = [(i, j) for i in range(n_in) for j in range(max(n_out, 1))]
        table = []
        for ph in phases:
            table += [(ph, 1)] * green + [(ph, 2)] * amber + [(ph, 0)] * allred
        for k in range(3 * len(table)):
            ph, colour = table[(k + off) % len(table)]
            for i in range(n_in):
                for j in range(max(n_out, 1)):
                    got = L.orc_signal_phase(green, amber, allred, off, n_in, n_out, i, j, k)
                    assert got == (colour if (i, j) == ph else 0), (n_in, n_out, k, i, j)
    # amber = 0 and n_out = 0 is the plan of reading R16
    for k in range(200):
        for r in range(4):
            assert L.orc_signal_phase(7, 0, 3, 5, 4, 0, r, 0, k) == L.orc_signal_green(7, 3, 5, 4, r, k)


def test_movement_phases_reduce_to_inbound_phases_where_every_node_has_one_exit():
    """n*m with m = 1 is reading R16's plan: on a chain of edges both controls give the same run."""
    sig = (np.full(7, 20), np.full(7, 4), np.arange(7) * 5)
    runs = []
    for ctrl in (W.CTRL_SIGNAL, W.CTRL_SIGNAL_NM):
        b = corridor(n_edges=6, length=300, departs=np.arange(40) * 3.0, ctrl=ctrl, sig=sig, steps=1500)
        runs.append(Oracle(b).step(1500, digests=True, check=1))
    assert (runs[0] == runs[1]).all()


def _crossings(b, steps, check=1):
    """Run and record (step k, vehicle, from edge, to edge, state before the step)."""
    o = Oracle(b)
    st = o.read_state()
    out = []
    for k in range(steps):
        o.step(1, check=check)
        after = o.read_state()
        moved = np.nonzero((st["status"] == 1) & (after["status"] == 1) & (after["edge"] != st["edge"]))[0]
        for i in moved:
            out.append((k, int(i), int(st["edge"][i]), int(after["edge"][i]), float(st["x"][i]), float(st["v"][i])))
        st_prev, st = st, after
    return o, out


def test_amber_and_movement_phases_on_a_grid():
    """Every crossing of a signalised node happens in the crosser's own phase -- looked up in an
    explicit timetable built here -- during its green, or during its amber and then only by a
    vehicle that could not have stopped: v^2 > 2 b (C - x) (reading R36).  Both kinds occur."""
    base = small_signal_grid(n_vehicles=1200, steps=900)
    b = W.with_controls(base, amber_steps=5)
    p = b["params"]
    ef, et = b["edge_from"], b["edge_to"]
    n_in = np.bincount(et, minlength=b["n_nodes"]); n_out = np.bincount(ef, minlength=b["n_nodes"])
    in_rank = np.zeros(len(ef), int); out_rank = np.zeros(len(ef), int)
    seen_in, seen_out = {}, {}
    for e in range(len(ef)):
        in_rank[e] = seen_in.get(int(et[e]), 0); seen_in[int(et[e])] = in_rank[e] + 1
        out_rank[e] = seen_out.get(int(ef[e]), 0); seen_out[int(ef[e])] = out_rank[e] + 1
    o, xs = _crossings(b, 900)
    greens = ambers = nm = 0
    for k, i, e, e2, x, v in xs:
        h = int(et[e]); ctrl = int(b["node_ctrl"][h])
        if ctrl not in (W.CTRL_SIGNAL, W.CTRL_SIGNAL_NM):
            continue
        g, r = int(b["sig_green_steps"][h]), int(b["sig_allred_steps"][h])
        Pd = g + p["amber_steps"] + r
        m = int(n_out[h]) if ctrl == W.CTRL_SIGNAL_NM else 1
        mine = in_rank[e] * m + (out_rank[e2] if ctrl == W.CTRL_SIGNAL_NM else 0)
        t = (k + int(b["sig_offset_steps"][h])) % (int(n_in[h]) * m * Pd)
        assert t // Pd == mine, (k, i, "crossed in somebody else's phase")
        pos = t % Pd
        assert pos < g + p["amber_steps"], (k, i, "crossed on red")
        nm += ctrl == W.CTRL_SIGNAL_NM
        if pos < g:
            greens += 1
        else:
            ambers += 1
            rem = float(b["edge_len_m"][e]) - x
            assert v * v > 2.0 * p["b"] * rem - 1e-3, (k, i, v, rem)
    assert greens > 200 and ambers >= 5 and nm > 50, (greens, ambers, nm)


def test_amber_stops_those_who_can_stop():
    """One vehicle, one signal at the end of a 600 m edge (cycle 100 steps: green [0, 60), amber
    [60, 70), red [70, 100)), departure time swept so that it meets the amber at every distance
    from the line.  Rule R36 from the recorded states: on amber it goes on iff v^2 > 2 b (C - x);
    a vehicle that could stop when the amber came up is still on the edge when the red begins."""
    b_ = P["b"]
    went = stopped = 0
    for depart in np.arange(0.0, 50.0, 1.5):
        sig = (np.full(3, 60), np.full(3, 30), np.zeros(3, int))
        b = corridor(n_edges=2, length=600, departs=(float(depart),), ctrl=W.CTRL_SIGNAL, sig=sig, steps=400,
                     params=dict(amber_steps=10))
        o = Oracle(b)
        st = o.read_state()
        could_stop_at_amber = None
        for k in range(400):
            o.step(1, check=1)
            after = o.read_state()
            pos = k % 100
            on_edge0 = st["status"][0] == 1 and st["edge"][0] == 0
            if on_edge0 and pos == 60:
                rem, v = 600.0 - float(st["x"][0]), float(st["v"][0])
                could_stop_at_amber = v * v < 2.0 * b_ * rem - 1e-3
            if on_edge0 and after["edge"][0] == 1:                       # crossed in step k
                assert pos < 70, (depart, k, "crossed on red")
                if pos >= 60:
                    rem, v = 600.0 - float(st["x"][0]), float(st["v"][0])
                    assert v * v > 2.0 * b_ * rem - 1e-3, (depart, k)
                    went += 1
                break
            if on_edge0 and pos == 69 and could_stop_at_amber:
                stopped += 1                                             # still there when the red begins
            st = after
    assert went >= 2 and stopped >= 2, (went, stopped)


# ------------------------------------------------------------------ STOP control

def test_stop_control_one_at_a_time_until_the_node_is_cleared():
    """"For stop controls our system allows just one vehicle at a time into the
    intersection and waits until the car has reached the next edge."  Reading R34, checked from the
    recorded states: whoever crosses a STOP node (a) has made a stop on its edge -- some earlier
    state within stop_dist of the line at no more than stop_speed; (b) does so only when the
    previous crosser of that node has its REAR past the node (x >= its length on the edge it
    entered, or it has left that edge); (c) alone in its step."""
    b = W.with_controls(W.config1())            # every node of config 1 becomes a STOP node
    b = W.with_trucks(b, share=0.2)
    p = b["params"]
    lens = np.asarray(p["type_len"])[b["veh_type"]]
    o = Oracle(b)
    st = o.read_state()
    stopped_on = {}            # vehicle -> edge on which it has made its stop
    holder = {}                # node -> (vehicle, edge it entered)
    n_cross = n_waited = 0
    for k in range(3600):
        act = np.nonzero(st["status"] == 1)[0]
        for i in act:
            e = int(st["edge"][i])
            if float(b["edge_len_m"][e]) - float(st["x"][i]) <= p["stop_dist"] and float(st["v"][i]) <= p["stop_speed"]:
                stopped_on[int(i)] = e
        o.step(1, check=1)
        after = o.read_state()
        moved = np.nonzero((st["status"] == 1) & (after["status"] == 1) & (after["edge"] != st["edge"]))[0]
        nodes = [int(b["edge_to"][st["edge"][i]]) for i in moved]
        assert len(set(nodes)) == len(nodes), (k, "two vehicles crossed one STOP node in one step")
        for i, h in zip(moved, nodes):
            i = int(i)
            assert stopped_on.get(i) == int(st["edge"][i]), (k, i, "crossed without having stopped")
            if h in holder:
                j, ej = holder[h]
                cleared = st["status"][j] != 1 or int(st["edge"][j]) != ej or float(st["x"][j]) >= lens[j]
                assert cleared, (k, i, j, "crossed while the node was held")
            holder[h] = (i, int(after["edge"][i]))
            n_cross += 1
        # somebody standing at a held node must be waiting
        for h, (j, ej) in holder.items():
            if st["status"][j] == 1 and int(st["edge"][j]) == ej and float(st["x"][j]) < lens[j]:
                n_waited += 1
        st = after
    assert n_cross > 500 and n_waited > 100
    assert after["n_arrived"] == b["n_vehicles"]
