"""Pins of the oracle against what the paper and the mathematics fix (no GPU).

Each test ties oracle/ts_oracle.c to something other than itself:
  P1  lone vehicle  -> closed-form integral of Eq. 7's free term (tests/golden/idm_free_road.txt)
  P2  platoon       -> equilibrium gap s_e = (s0+vT)/sqrt(1-(v/v0)^4) (tests/golden/idm_equilibrium_gap.txt)
  P3  standing queue at a red line -> fronts s0 + veh_len apart
  I1-I8 invariants, P4 brute force (orc_step check=2), P5 degenerate cases
  scalar pieces: Eq. 7 in fp64 at a grid of points, signal round robin, speed code grid.
"""
import math
import os

import numpy as np
import pytest

from oracle import Oracle, OracleError, idm, lib
from paper_1807_01148_b200 import workload as W

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")
P = W.DEFAULT_PARAMS


def _rows(name):
    out = []
    for line in open(os.path.join(GOLDEN, name)):
        if line.strip() and not line.startswith("#"):
            out.append([float(t) for t in line.split()])
    return out


def corridor(n_edges=1, length=4000, lanes=1, vlim=15.0, departs=(0.0,), v0_mult=None,
             ctrl=W.CTRL_FREE, steps=400, params=None, sig=None, route_len=None, mand=None):
    """A straight chain of `n_edges` edges 0->1->...; every vehicle drives the first
    `route_len` edges."""
    N = n_edges + 1
    ef, et = np.arange(n_edges), np.arange(1, n_edges + 1)
    V = len(departs)
    rl = route_len or n_edges
    route_off = np.arange(V + 1) * rl
    route_edges = np.tile(np.arange(rl), V)
    g, r, o = sig if sig else (None, None, None)
    return W.make_bundle("corridor", N, ef, et, np.full(n_edges, length), np.full(n_edges, lanes),
                         np.full(n_edges, vlim), np.full(N, ctrl), route_off, route_edges,
                         np.asarray(departs, np.float32), steps, g, r, o, v0_mult, mand, params)


# ------------------------------------------------------------------ scalar pieces

def test_idm_matches_eq7_in_fp64():
    """Eq. 7 evaluated in fp64 at a grid of points; fp32 oracle within 1e-5 rel."""
    a, b, T, s0 = P["a"], P["b"], P["T"], P["s0"]
    for v in (0.0, 3.3, 12.0, 14.9):
        for s in (0.7, 2.0, 9.0, 55.5, 120.0):
            for dv in (-5.0, 0.0, 4.0):
                v0 = 15.0
                sstar = s0 + max(0.0, T * v + v * dv / (2 * math.sqrt(a * b)))
                want = a * (1 - (v / v0) ** 4 - (sstar / max(s, 0.5)) ** 2)
                got = idm(P, v, v0, True, s, dv)
                assert got == pytest.approx(want, rel=2e-5, abs=2e-5)
        assert idm(P, v, 15.0, False, 0, 0) == pytest.approx(a * (1 - (v / 15.0) ** 4), abs=1e-6)


def test_idm_signs():
    """A plausible mistake (wrong sign of dv, s and s* swapped) fails here."""
    assert idm(P, 10, 15, True, 30, +5) < idm(P, 10, 15, True, 30, 0) < idm(P, 10, 15, True, 30, -5)
    assert idm(P, 10, 15, True, 10, 0) < idm(P, 10, 15, True, 40, 0)
    assert idm(P, 0, 15, True, 2.0, 0) == pytest.approx(0.0, abs=1e-6)   # s = s0 at rest: equilibrium


def test_speed_code_grid():
    L = lib()
    assert L.orc_speed_code(0.0) == 1 and L.orc_speed_decode(1) == 0.0
    for q in range(0, 255):
        assert L.orc_speed_code(q * 0.25) == q + 1
        assert L.orc_speed_decode(q + 1) == q * 0.25
    assert L.orc_speed_code(1000.0) == 255
    assert L.orc_speed_code(0.124) == 1 and L.orc_speed_code(0.126) == 2   # round to nearest


def test_signal_round_robin():
    """round robin over inbound edges; never two greens, each gets `green` steps."""
    L = lib()
    green, allred, n_in, off = 7, 3, 4, 5
    cyc = n_in * (green + allred)
    count = np.zeros(n_in, int)
    for k in range(cyc):
        g = [L.orc_signal_green(green, allred, off, n_in, r, k) for r in range(n_in)]
        assert sum(g) <= 1
        count += np.array(g)
    assert (count == green).all()
    assert L.orc_signal_green(green, allred, 0, n_in, 0, 0) == 1
    assert L.orc_signal_green(green, allred, 0, n_in, 0, green) == 0
    assert L.orc_signal_green(green, allred, 0, n_in, 1, green + allred) == 1
    assert L.orc_signal_green(green, allred, off, n_in, 2, 3 * cyc + 11) == L.orc_signal_green(green, allred, off, n_in, 2, 11)


# ------------------------------------------------------------------ P1 lone vehicle

def _t_closed(u, v0, a):
    return (v0 / a) * (0.25 * math.log((1 + u) / (1 - u)) + 0.5 * math.atan(u))


def test_p1_golden_values_are_the_closed_form():
    for v0, a, u, t in _rows("idm_free_road.txt"):
        assert _t_closed(u, v0, a) == pytest.approx(t, abs=1e-3)


@pytest.mark.parametrize("v0", [11.0, 15.0, 29.0])
def test_p1_lone_vehicle(v0):
    """One vehicle, one long edge, from rest: v(t) follows the integral of Eq. 7's free term
    within 0.10 m/s at every step (explicit Euler at dt = 0.5), monotone, never above v0."""
    b = corridor(length=30000, vlim=v0, steps=400)
    o = Oracle(b)
    prev = 0.0
    worst = 0.0
    for k in range(1, 241):
        o.step(1, check=1)
        st = o.read_state()
        v = float(st["v"][0])
        if st["status"][0] != 1:
            continue
        t = (k - 1) * P["dt"]            # inserted at the end of step 1 with v = 0
        lo, hi = 0.0, 1.0 - 1e-12        # invert t(u) by bisection
        for _ in range(80):
            mid = 0.5 * (lo + hi)
            if _t_closed(mid, v0, P["a"]) < t:
                lo = mid
            else:
                hi = mid
        worst = max(worst, abs(v - lo * v0))
        assert v >= prev - 1e-6 and v <= v0
        prev = v
    assert worst <= 0.10, worst
    assert prev > 0.99 * v0


def test_p1_golden_times():
    """The simulated vehicle reaches u = 0.5, 0.9, 0.99 within one step of the golden times."""
    for v0, a, u, t in _rows("idm_free_road.txt"):
        o = Oracle(corridor(length=30000, vlim=v0))
        reached = None
        for k in range(1, 200):
            o.step(1)
            if o.read_state()["v"][0] >= u * v0:
                reached = (k - 1) * P["dt"]
                break
        assert reached is not None and abs(reached - t) <= 0.75, (u, reached, t)


# ------------------------------------------------------------------ P2 platoon equilibrium

@pytest.mark.parametrize("row", _rows("idm_equilibrium_gap.txt")[:2])
def test_p2_platoon_gap(row):
    v0, v, s0, T, s_e = row
    assert (s0 + v * T) / math.sqrt(1 - (v / v0) ** 4) == pytest.approx(s_e, abs=1e-3)
    b = corridor(length=30000, vlim=v0, departs=(0.0, 10.0), v0_mult=np.array([v / v0, 1.0]))
    o = Oracle(b)
    o.step(2000, check=1)
    st = o.read_state()
    assert st["v"][0] == pytest.approx(v, abs=1e-3)
    perceived = float(st["cell"][0]) - P["veh_len"] - float(st["x"][1])
    true_gap = float(st["x"][0]) - P["veh_len"] - float(st["x"][1])
    assert abs(perceived - s_e) <= 0.01, (perceived, s_e)
    assert s_e - 1e-2 <= true_gap < s_e + 1.0
    assert st["v"][1] == pytest.approx(v, abs=0.01)


def test_p2_off_grid_speed():
    """Leader speed off the 0.25 m/s grid: small limit cycle, true gap within 1.5 m of s_e."""
    v0, v = 15.0, 12.3
    s_e = (P["s0"] + v * P["T"]) / math.sqrt(1 - (v / v0) ** 4)
    o = Oracle(corridor(length=60000, vlim=v0, departs=(0.0, 10.0), v0_mult=np.array([v / v0, 1.0])))
    o.step(2000)
    for _ in range(20):
        o.step(1)
        st = o.read_state()
        gap = float(st["x"][0]) - P["veh_len"] - float(st["x"][1])
        assert abs(gap - s_e) <= 1.5, (gap, s_e)


# ------------------------------------------------------------------ P3 standing queue

def test_p3_standing_queue_at_red():
    """Vehicles released toward a permanently red line stop with the first front about s0
    short of the line and successive fronts veh_len + s0 = 7 m apart (+-1 m: one cell)."""
    n = 6
    N = 3
    sig = (np.full(N, 1), np.full(N, 1_000_000), np.full(N, 1))     # green only at k = 10^6
    b = corridor(n_edges=2, length=600, departs=np.arange(n) * 4.0, ctrl=W.CTRL_SIGNAL, sig=sig,
                 steps=2000)
    o = Oracle(b)
    o.step(1600, check=1)
    st = o.read_state()
    assert (st["status"] == 1).all() and (st["edge"] == 0).all()
    assert (st["v"] < 0.02).all()
    x = st["x"].astype(float)
    assert 600 - P["s0"] - 1.0 <= x[0] <= 600 - P["s0"] + 0.5
    d = x[:-1] - x[1:]
    assert (np.abs(d - (P["veh_len"] + P["s0"])) <= 1.0).all(), d
    # and nobody ever crossed on red
    assert o.read_edge_stats()["entered"][1] == 0
