"""Pins of the oracle's section 6.3.4 accumulators (Eq. 8 CO, Eq. 9 fuel;
SURVEY.md 8(f) row 2) against what the paper's formulas fix (no GPU).

  rates      Eq. 8 / Eq. 9 at points worked by hand from the printed coefficients
             (tests/golden/emission_rates.txt), sign and special cases
  idle       a queue standing at a red line accumulates 0.586 g/s of CO (Eq. 8 at 0 mph) and
             0.666 mL/s of fuel (Eq. 9 at v = 0)
  cruise     a lone vehicle that has reached 50 mph accumulates 0.216 g/s (the vertex term of
             Eq. 8 vanishes) and Eq. 9's polynomial in v alone
  quadrature a lone vehicle accelerating from rest: totals against an fp64 fine-step integration
             of Eq. 7's free-road ODE with Eq. 8 / Eq. 9 as integrands
  invariants nothing for a vehicle that never drove, monotone growth, bounds from the time spent
             on the road, and the traffic itself is untouched by the accumulators
"""
import os

import numpy as np
import pytest

from oracle import Oracle, co_rate, fuel_rate
from paper_1807_01148_b200 import workload as W
from test_oracle_pins import corridor

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")
MPH = 3600.0 / 1609.344          # miles per hour in one m/s
EM = dict(emissions=1)


def test_rates_match_the_papers_formulas_at_hand_worked_points():
    n = 0
    for line in open(os.path.join(GOLDEN, "emission_rates.txt")):
        if not line.strip() or line.startswith("#"):
            continue
        kind, speed, acc, want = line.split()
        speed, acc, want = float(speed), float(acc), float(want)
        got = co_rate(speed / MPH) if kind == "co" else fuel_rate(speed, acc)
        assert got == pytest.approx(want, rel=2e-5), line
        n += 1
    assert n == 10


def test_rate_shapes():
    """A dropped or mis-signed term fails here."""
    # Eq. 8 is a parabola in mph with its minimum where 0.0056 + 0.00052 (vm - 50) = 0
    vm_min = 50 - 0.0056 / 0.00052
    grid = np.linspace(0, 90, 181)
    vals = [co_rate(v / MPH) for v in grid]
    assert abs(grid[int(np.argmin(vals))] - vm_min) <= 0.5
    assert min(vals) > 0.18
    # Eq. 9: P_ea only for a > 0; the a*v term acts in both directions
    assert fuel_rate(15, 0.5) - fuel_rate(15, 0) > 0.072 * 1.680 * 0.5 * 15          # + P_ea
    assert fuel_rate(15, 0) - fuel_rate(15, -0.1) == pytest.approx(0.072 * 1.680 * 0.1 * 15, rel=1e-4)
    assert fuel_rate(0, 3.0) == pytest.approx(0.666, rel=1e-6)                        # every term carries v
    assert fuel_rate(25, -5.0) == pytest.approx(0.666, rel=1e-6)                      # floor (R29)


def test_idle_queue_at_red():
    n, N = 5, 3
    sig = (np.full(N, 1), np.full(N, 1_000_000), np.full(N, 1))
    b = corridor(n_edges=2, length=600, departs=np.arange(n) * 4.0, ctrl=W.CTRL_SIGNAL, sig=sig,
                 steps=3000, params=EM)
    o = Oracle(b)
    o.step(1800, check=1)
    e0 = o.read_emissions()
    assert (o.read_state()["v"] < 0.02).all()
    o.step(1000, check=1)                      # 500 s standing
    e1 = o.read_emissions()
    assert (e1["co_g"] - e0["co_g"]) == pytest.approx(np.full(n, 0.586 * 500), rel=3e-3)
    assert (e1["fuel_ml"] - e0["fuel_ml"]) == pytest.approx(np.full(n, 0.666 * 500), rel=3e-3)


def test_cruise_at_50_mph():
    v0 = 50.0 / MPH                            # 22.352 m/s
    b = corridor(length=60000, vlim=v0, steps=4000, params=EM)
    o = Oracle(b)
    o.step(1000)                               # 500 s: v has converged to v0
    v = float(o.read_state()["v"][0])
    assert v == pytest.approx(v0, abs=2e-3)
    e0 = o.read_emissions()
    o.step(400)                                # 200 s of cruising
    e1 = o.read_emissions()
    assert float(e1["co_g"][0] - e0["co_g"][0]) == pytest.approx(0.216 * 200, rel=2e-3)
    f = 0.666 + 0.072 * (0.269 * v0 + 0.0171 * v0 ** 2 + 0.000672 * v0 ** 3)
    assert float(e1["fuel_ml"][0] - e0["fuel_ml"][0]) == pytest.approx(f * 200, rel=3e-3)


@pytest.mark.parametrize("v0", [13.0, 29.0])
def test_acceleration_run_against_fp64_quadrature(v0):
    """dv/dt = a (1 - (v/v0)^4) (Eq. 7, free road) integrated in fp64 with RK4 at 1 ms, Eq. 8 and
    Eq. 9 (with that acceleration, P_ea included) as integrands.  The simulator's Euler step of
    0.5 s is within 0.10 m/s of that trajectory (pin P1); the totals agree to a few per cent."""
    a, T = W.DEFAULT_PARAMS["a"], 40.0

    def acc(v):
        return a * (1 - (v / v0) ** 4)

    def co(v):
        vm = v * MPH
        return -0.064 + 0.0056 * vm + 0.00026 * (vm - 50) ** 2

    def fuel(v):
        ac = acc(v)
        br = 0.269 * v + 0.0171 * v ** 2 + 0.000672 * v ** 3 + 1.680 * ac * v
        if ac > 0:
            br += 0.79296 * ac * ac * v
        return 0.666 + 0.072 * max(br, 0.0)

    h, v, tot_co, tot_fuel = 1e-3, 0.0, 0.0, 0.0
    for _ in range(int(T / h)):
        k1 = acc(v); k2 = acc(v + 0.5 * h * k1); k3 = acc(v + 0.5 * h * k2); k4 = acc(v + h * k3)
        vn = v + h * (k1 + 2 * k2 + 2 * k3 + k4) / 6
        tot_co += 0.5 * h * (co(v) + co(vn))
        tot_fuel += 0.5 * h * (fuel(v) + fuel(vn))
        v = vn
    b = corridor(length=60000, vlim=v0, steps=200, params=EM)
    o = Oracle(b)
    o.step(int(T / 0.5) + 1)                   # inserted at step 1, then T seconds of driving
    e = o.read_emissions()
    assert float(e["co_g"][0]) == pytest.approx(tot_co, rel=0.02)
    assert float(e["fuel_ml"][0]) == pytest.approx(tot_fuel, rel=0.015)
    # the engine-drag term matters in this run: without P_ea the total would be out of tolerance
    assert tot_fuel > 1.06 * (0.666 * T)


def test_invariants_on_config1():
    b = W.by_name("cfg1")
    b = dict(b, params=dict(b["params"], emissions=1))
    o = Oracle(b)
    plain = Oracle(W.by_name("cfg1"))
    prev = o.read_emissions()
    for _ in range(12):
        d1 = o.step(300, digests=True, check=1)
        d0 = plain.step(300, digests=True)
        assert (d1 == d0).all()                # the accumulators never feed back into the traffic
        e, st = o.read_emissions(), o.read_state()
        assert (e["co_g"] >= prev["co_g"]).all() and (e["fuel_ml"] >= prev["fuel_ml"]).all()
        never = st["status"] == 0
        assert (e["co_g"][never] == 0).all() and (e["fuel_ml"][never] == 0).all()
        prev = e
    st = o.read_state()
    done = st["status"] == 2
    assert done.all()
    secs = (st["arrive_step"] - st["insert_step"]).astype(float) * 0.5
    co, fuel = prev["co_g"].astype(float), prev["fuel_ml"].astype(float)
    # Eq. 8 lies in [0.186, 0.586] g/s for 0..15 m/s; Eq. 9 is at least the idle rate and, with
    # a <= 1 m/s^2 and v <= 15 m/s, at most 0.666 + 0.072 (10.15 + 25.2 + 11.9) = 4.07 mL/s
    assert (co >= 0.186 * secs * 0.999).all() and (co <= 0.586 * secs * 1.001).all()
    assert (fuel >= 0.666 * secs * 0.999).all() and (fuel <= 4.07 * secs).all()
    assert plain.read_emissions()["co_g"].sum() == 0          # off unless asked for
