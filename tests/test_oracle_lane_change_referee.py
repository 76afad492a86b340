"""A referee for the lane-change rule (step 2d) and for the
gap to a leader beyond the node (Eq. 7 with E3's "across the node" gap).

The referee below re-derives, in Python and fp64 and from the RULE TEXT of DESIGN.md section 2 (not
from oracle/ts_oracle.c), the decision of every vehicle whose turn it is at every step of dense
multi-lane scenarios -- eligibility, gap acceptance G1 (lead gap >= s0), G2 (lag gap >= s0 and >=
the kinematic bound (vF + 0.125 + a dt / 2) dt), G3 (the new follower's braking >= -b_safe), the
mandatory rule, the veto of a discretionary move into a lane that does not continue, and the MOBIL
incentive (a~_c - a_c) + p (a~_F - a_F) > threshold -- from the state BEFORE the step as the
traffic atlas shows it (cell index, speed on the 0.25 m/s grid), and compares with the lane the
oracle gives the vehicle AFTER the step.  A decision whose margin is below 2e-3 in fp64 is left out
(fp32 against fp64), and each scenario must contain decisions that only one sub-rule decides:
  * the politeness term flips the verdict (both ways across p = 0.2 and p = 0.5),
  * G2 rejects through its kinematic bound although lag gap >= s0,
  * G3 rejects although G1 and G2 pass,
  * a mandatory change happens at the first eligible turn inside mand_dist (and discretionary
    rules apply before), a discretionary move into a dropped lane is vetoed inside mand_dist.
Mutations of the oracle that these tests catch (each tried by hand while writing them): dropping
E4's `m` term, `>= -b_safe` -> `>= +b_safe` or `<=`, dropping `politeness * d2`, `l >= lanes_e2`
-> `>` (and the same in the veto), dropping `+ cL2` from the across-the-node gap, `cF + 1` -> `cF` in the
lag gap and in a_F's gap, a_c against a leader that is beyond the node, G1 against 0 instead of s0.
"""
import math

import numpy as np
import pytest

from oracle import Oracle
from paper_1807_01148_b200 import workload as W
from test_oracle_invariants import small_signal_grid
from test_oracle_pins import _rows, corridor

EPS = 2e-3


def _idm64(p, v, v0, has, s=0.0, dv=0.0, a=None):
    """Eq. 7 in fp64 with readings R1, R2, R8; `a` = the subject vehicle's
    acceleration ability where vehicle types differ."""
    a = p["a"] if a is None else a
    free = 1.0 - (v / v0) ** 4
    if not has:
        return a * free
    sstar = p["s0"] + max(0.0, v * p["T"] + v * dv / (2.0 * math.sqrt(a * p["b"])))
    return a * (free - (sstar / max(s, 0.5)) ** 2)


def _seen_speed(v):
    """What the atlas shows of a speed (reading R5): 0.25 m/s grid, round half up, capped."""
    q = np.float32(v) * np.float32(4.0) + np.float32(0.5)
    return min(254, int(q)) * 0.25


class Referee:
    def __init__(self, bundle):
        self.b = bundle
        self.p = p = bundle["params"]
        # vehicle types: per vehicle its length, acceleration ability and speed cap
        V = bundle["n_vehicles"]
        ty = np.zeros(V, int) if bundle.get("veh_type") is None else np.asarray(bundle["veh_type"], int)
        if p.get("n_types", 0):
            self.len_of = np.asarray(p["type_len"], float)[ty]
            self.a_of = np.asarray(p["type_a"], float)[ty]
            self.vmax_of = np.asarray(p["type_vmax"], float)[ty]
        else:
            self.len_of, self.a_of, self.vmax_of = np.full(V, p["veh_len"]), np.full(V, p["a"]), np.full(V, np.inf)
        self.tally = dict(turns=0, accepted=0, skipped=0, polite_flips_to_yes=0, polite_flips_to_no=0,
                          g1_rejects=0, g2_kinematic_rejects=0, g3_rejects=0, mandatory=0, vetoes_of_a_wanted_move=0,
                          discretionary_before_mand_dist=0, with_lag=0, with_lead=0)

    def lanes_of(self, st):
        """(edge, lane) -> sorted array of (cell, vehicle) of the ACTIVE vehicles, from raw state."""
        act = np.nonzero(st["status"] == 1)[0]
        out = {}
        for i in act:
            out.setdefault((int(st["edge"][i]), int(st["lane"][i])), []).append((int(st["cell"][i]), int(i)))
        for key in out:
            out[key].sort()
        return out

    def decide(self, st, lanes, i, k):
        """Returns None (not this vehicle's turn), or (new lane, margins) by the rule text."""
        b, p = self.b, self.p
        e, l = int(st["edge"][i]), int(st["lane"][i])
        x, v = float(st["x"][i]), float(st["v"][i])
        C = int(b["edge_len_m"][e])
        n_lanes = int(b["edge_lanes"][e])
        dt, a, length = p["dt"], float(self.a_of[i]), float(self.len_of[i])
        H, Hb = p["lookahead_cells"], p["lookback_cells"]
        margins = []
        if p["lc_period"] == 0 or n_lanes < 2:
            return None
        lt = l + (1 if k % 2 == 0 else -1)
        if not (0 <= lt < n_lanes) or ((k >> 1) + i) % p["lc_period"] != 0 or x < p["entry_zone_cells"]:
            return None
        reach = x + (v + a * dt) * dt
        if abs(reach - C) < EPS:
            return "skip"
        if not reach < C:
            return None
        c = int(math.floor(x))
        route = b["route_edges"][int(b["route_off"][i]):int(b["route_off"][i + 1])]
        r = int(st["route_idx"][i])
        last = r == len(route) - 1
        lanes2 = 0 if last else int(b["edge_lanes"][route[r + 1]])
        v0 = min(float(np.float32(b["v0_mult"][i]) * np.float32(b["edge_vlim"][e])), float(self.vmax_of[i]))
        vlim = float(b["edge_vlim"][e])
        # neighbours in the target lane and the own leader, all on this edge only
        tl = lanes.get((e, lt), [])
        ahead = [(cc, j) for cc, j in tl if c <= cc <= min(C - 1, c + H)]
        behind = [(cc, j) for cc, j in tl if max(0, c - Hb) <= cc <= c - 1]
        own = [(cc, j) for cc, j in lanes.get((e, l), []) if c < cc <= min(C - 1, c + H)]
        has_Lt, has_F, lead_on_edge = bool(ahead), bool(behind), bool(own)
        cLt = vLt = s_Lt = cF = vF = s_lag = len_Lt = 0.0
        a_lag, v0_lag = a, vlim
        if has_Lt:
            cLt, j = ahead[0]
            vLt = _seen_speed(st["v"][j])
            len_Lt = float(self.len_of[j])
            s_Lt = cLt - len_Lt - x                       # the LEADER's length
        if has_F:
            cF, j = behind[-1]
            vF = _seen_speed(st["v"][j])
            s_lag = x - length - (cF + 1)                 # the changer's own length
            a_lag, v0_lag = float(self.a_of[j]), min(vlim, float(self.vmax_of[j]))
        t = self.tally
        t["turns"] += 1
        t["with_lag"] += has_F
        t["with_lead"] += has_Lt

        def cmp_ge(lhs, rhs):
            margins.append(lhs - rhs)
            return lhs >= rhs

        if has_Lt and not cmp_ge(s_Lt, p["s0"]):                               # G1
            t["g1_rejects"] += 1
            return l, margins
        aF_new = 0.0
        if has_F:
            bound = (vF + 0.125 + 0.5 * a_lag * dt) * dt                        # G2 with E4
            ok_s0 = cmp_ge(s_lag, p["s0"])
            ok_kin = cmp_ge(s_lag, bound)
            if not (ok_s0 and ok_kin):
                if ok_s0:
                    t["g2_kinematic_rejects"] += 1
                return l, margins
            aF_new = _idm64(p, vF, v0_lag, True, s_lag, vF - v, a_lag)          # G3
            if not cmp_ge(aF_new, -p["b_safe"]):
                t["g3_rejects"] += 1
                return l, margins
        rem = C - x                                                            # G4
        mand = float(b["mand_dist_m"][i])
        inside = rem <= mand
        margins.append(rem - mand)
        at_c = _idm64(p, v, v0, has_Lt, s_Lt, v - vLt, a)
        a_c = _idm64(p, v, v0, True, own[0][0] - float(self.len_of[own[0][1]]) - x,
                     v - _seen_speed(st["v"][own[0][1]]), a) if lead_on_edge else _idm64(p, v, v0, False, a=a)
        inc_self = at_c - a_c
        inc = inc_self
        if has_F:
            a_F = _idm64(p, vF, v0_lag, has_Lt, cLt - len_Lt - (cF + 1), vF - vLt, a_lag)
            inc = inc_self + p["politeness"] * (aF_new - a_F)
        if not last and l >= lanes2 and lt < l and inside:
            t["mandatory"] += 1
            return lt, margins
        if not last and lt >= lanes2 and inside:
            if inc > p["lc_threshold"] + EPS:
                t["vetoes_of_a_wanted_move"] += 1
            return l, margins
        margins.append(inc - p["lc_threshold"])
        yes = inc > p["lc_threshold"]
        if has_F and abs(inc_self - p["lc_threshold"]) > EPS and (inc_self > p["lc_threshold"]) != yes:
            t["polite_flips_to_yes" if yes else "polite_flips_to_no"] += 1
        if not last and l >= lanes2 and lt < l:
            t["discretionary_before_mand_dist"] += 1
        return (lt if yes else l), margins

    def run(self, steps, check=1):
        o = Oracle(self.b)
        st = o.read_state()
        for k in range(steps):
            lanes = self.lanes_of(st)
            want = {}
            for i in np.nonzero(st["status"] == 1)[0]:
                d = self.decide(st, lanes, int(i), k)
                if d == "skip" or (d is not None and any(abs(m) < EPS for m in d[1])):
                    self.tally["skipped"] += 1
                    want[int(i)] = None
                else:
                    want[int(i)] = int(st["lane"][i]) if d is None else d[0]
            o.step(1, check=check)
            after = o.read_state()
            for i, lane in want.items():
                if lane is None or after["status"][i] != 1 or after["edge"][i] != st["edge"][i]:
                    continue
                assert int(after["lane"][i]) == lane, (
                    f"step {k} vehicle {i}: oracle lane {int(after['lane'][i])}, rule text says {lane} "
                    f"(from lane {int(st['lane'][i])}, x={float(st['x'][i])}, v={float(st['v'][i])})")
                self.tally["accepted"] += lane != int(st["lane"][i])
            st = after
        return self.tally


def _platoon_scenario(politeness, seed):
    """Three lanes over two long edges, then one lane (so that lanes 1 and 2 must be left inside
    mand_dist): slow and fast vehicles released close together -- many changes with a lag vehicle
    near by, so that politeness, G2 and G3 get to decide."""
    rng = np.random.default_rng(seed)
    V = 260
    lanes = np.array([3, 3, 1])
    length = np.array([900, 700, 400])
    ef, et = np.arange(3), np.arange(1, 4)
    route_off = np.arange(V + 1) * 3
    route_edges = np.tile(np.arange(3), V)
    depart = np.sort(rng.random(V) * 500.0)
    v0m = rng.choice([0.35, 0.6, 1.0, 1.15], V, p=[0.2, 0.2, 0.4, 0.2])
    mand = rng.uniform(60.0, 350.0, V)
    return W.make_bundle("platoons", 4, ef, et, length, lanes, np.full(3, 17.0), np.zeros(4), route_off,
                         route_edges, depart, 1400, v0_mult=v0m, mand_dist_m=mand,
                         params=dict(politeness=politeness))


@pytest.mark.parametrize("politeness", [0.2, 0.5])
def test_every_lane_change_decision_in_dense_platoons(politeness):
    t = Referee(_platoon_scenario(politeness, 5)).run(1400)
    assert t["turns"] > 3000 and t["accepted"] > 100 and t["skipped"] < 0.05 * t["turns"], t
    assert t["with_lag"] > 500 and t["with_lead"] > 500, t
    assert t["polite_flips_to_no"] >= 3, t            # the follower's loss vetoes a move the changer wants
    assert t["g2_kinematic_rejects"] >= 3, t          # lag gap >= s0 but below the kinematic bound
    assert t["g3_rejects"] >= 3, t                    # gaps fine, but the new follower would brake harder than b_safe
    assert t["mandatory"] >= 20 and t["discretionary_before_mand_dist"] >= 20, t
    assert t["vetoes_of_a_wanted_move"] >= 3, t


def test_follower_terms_decide_under_magnified_politeness():
    """p = 8 (unphysical, legal): the new follower's present acceleration a_F -- its gap to Lt is
    cLt - len - (cF + 1) -- and its acceleration behind the changer weigh eight times the changer's
    own gain, so a slip of one cell in either follower gap changes verdicts here."""
    t = Referee(_platoon_scenario(8.0, 1)).run(1400)
    assert t["polite_flips_to_no"] >= 50 and t["skipped"] < 0.05 * t["turns"], t


def test_every_lane_change_decision_on_a_signalised_grid():
    """Queues at signals, 1-3 lanes, lanes that end at the next node (mandatory changes, vetoes)."""
    b = small_signal_grid(n_vehicles=1200, steps=800)
    t = Referee(b).run(800)
    assert t["turns"] > 2000 and t["mandatory"] >= 10 and t["g1_rejects"] >= 10, t
    # the politeness term decides both ways here: it vetoes moves the changer wants, and (rarely:
    # the changer is faster than the follower's present leader) it tips a move over the threshold
    assert t["polite_flips_to_no"] >= 3 and t["polite_flips_to_yes"] >= 1, t
    assert t["g2_kinematic_rejects"] >= 3 and t["g3_rejects"] >= 3 and t["vetoes_of_a_wanted_move"] >= 3, t
    assert t["skipped"] < 0.05 * t["turns"], t


def test_mandatory_change_happens_at_the_first_eligible_turn_inside_mand_dist():
    """One vehicle in lane 1 of a 2-lane edge whose successor has one lane, nobody else around:
    before C - x <= mand_dist the discretionary rule sees no incentive (empty road both sides) and
    it stays; at the FIRST turn with C - x <= mand_dist (odd k: towards the kerb) it moves.  A
    second vehicle in lane 0 with a slow leader ahead wants lane 1 (incentive > threshold) but is
    refused inside mand_dist, because lane 1 does not continue."""
    p = W.DEFAULT_PARAMS
    lanes = np.array([2, 2, 1])
    length = np.array([3000, 900, 300])
    ef, et = np.arange(3), np.arange(1, 4)
    # id 0: slow leader (stays in lane 0); id 1: overtakes it on edge 0 -> lane 1; both continue
    V = 2
    b = W.make_bundle("mand", 4, ef, et, length, lanes, np.full(3, 15.0), np.zeros(4), np.arange(V + 1) * 3,
                      np.tile(np.arange(3), V), np.array([0.0, 14.0]), 1200, v0_mult=np.array([0.5, 1.0]),
                      mand_dist_m=np.array([120.0, 230.0]))
    o = Oracle(b)
    st = o.read_state()
    went_left = back_at = None
    for k in range(1200):
        o.step(1, check=2)
        after = o.read_state()
        if went_left is None and after["lane"][1] == 1:
            went_left = k
        if went_left is not None and back_at is None and st["lane"][1] == 1 and after["lane"][1] == 0 and after["edge"][1] == st["edge"][1]:
            back_at = k
            x = float(st["x"][1]); e = int(st["edge"][1])
            assert e == 1                                            # the edge before the lane drop
            assert length[e] - x <= 230.0                           # inside its mand_dist ...
            assert k % 2 == 1 and ((k >> 1) + 1) % p["lc_period"] == 0   # ... on one of its turns to the right
            # ... and the first such turn: the previous turn (4 pairs of steps = 8 steps earlier) was outside
            v_then = float(st["v"][1])
            assert length[e] - (x - 8 * 0.5 * v_then) > 230.0 - 1.0
        st = after
    assert went_left is not None and back_at is not None
    assert o.counters()["lc_mandatory"] == 1


@pytest.mark.parametrize("row", _rows("idm_equilibrium_gap.txt")[:2])
def test_p2_equilibrium_gap_with_the_leader_beyond_the_node(row):
    """P2 again (tests/golden/idm_equilibrium_gap.txt, s_e = (s0 + vT)/sqrt(1 - (v/v0)^4)), on a
    chain of 300 m edges: whenever the pair straddles a node the follower sees its leader on the
    NEXT edge, and the gap it acts on is ((C - x) + cL2) - len (E3).  In equilibrium that perceived
    gap must equal s_e just as on one long edge; a slip in the across-the-node formula would make
    the follower brake or close up every 300 m."""
    v0, v, s0, T, s_e = row
    p = W.DEFAULT_PARAMS
    n_edges = 60
    b = corridor(n_edges=n_edges, length=300, vlim=v0, departs=(0.0, 10.0), v0_mult=np.array([v / v0, 1.0]), steps=2600)
    o = Oracle(b)
    o.step(2000, check=1)
    straddling = same_edge = 0
    for _ in range(400):
        o.step(1, check=1)
        st = o.read_state()
        if st["status"][0] != 1 or st["status"][1] != 1:
            break
        x_f, e_f, e_l = float(st["x"][1]), int(st["edge"][1]), int(st["edge"][0])
        if e_l == e_f:
            gap = float(st["cell"][0]) - p["veh_len"] - x_f
            same_edge += 1
        else:
            assert e_l == e_f + 1
            gap = ((300.0 - x_f) + float(st["cell"][0])) - p["veh_len"]
            straddling += 1
        assert abs(gap - s_e) <= 0.01, (gap, s_e, e_l == e_f)
        assert st["v"][1] == pytest.approx(v, abs=0.01)
    assert straddling >= 20 and same_edge >= 100
