"""Parity of the CUDA path against the oracle for SURVEY.md 8(f) rows 3 and 4: vehicle types
(reading R31) and the control variants of PAPER.md:402 (R34 STOP with a
persistent node owner, R35 one signal phase per movement, R36 amber).  Bit-exact at every step
(digests), in the final state and in the edge statistics, in both launch modes and under
different slot orders; plus the multi-step digest on many slots per thread."""
import numpy as np
import pytest

from paper_1807_01148_b200 import workload as W
from test_gpu_parity import _compare
from test_oracle_invariants import small_signal_grid
from test_oracle_pins import corridor

pytestmark = pytest.mark.gpu

TRUCKS = dict(n_types=2, type_len=(5.0, 12.0, 0, 0), type_a=(1.0, 0.5, 0, 0), type_vmax=(1000.0, 14.0, 0, 0),
              insert_clear_cells=14)


@pytest.mark.parametrize("mode", [1, 0])
def test_trucks_on_the_signal_grid(mode):
    b = W.with_trucks(small_signal_grid(), share=0.3)
    _compare(b, b["steps"], mode)


@pytest.mark.parametrize("mode", [1, 0])
def test_control_variants_on_the_signal_grid(mode):
    b = W.with_controls(small_signal_grid(), amber_steps=5)      # STOP, n*m phases, amber
    assert set(np.unique(b["node_ctrl"])) >= {W.CTRL_STOP, W.CTRL_SIGNAL, W.CTRL_SIGNAL_NM}
    _compare(b, b["steps"], mode)


@pytest.mark.parametrize("options", [dict(sort_period=1), dict(sort_period=7, threads=128), dict(sort_period=0),
                                     dict(adaptive_chunk=37, adaptive_above=0), dict(threads=1024)])
def test_trucks_and_controls_do_not_depend_on_slot_order(options):
    b = W.with_controls(W.with_trucks(small_signal_grid(), share=0.25), amber_steps=3)
    b = dict(b, params=dict(b["params"], emissions=1))
    _compare(b, b["steps"], 1, **options)


def test_stop_control_everywhere(cfg1):
    b = W.with_trucks(W.with_controls(cfg1), share=0.2)           # every node of config 1 is a STOP node
    st = _compare(b, b["steps"], 1, chunk=900)
    assert st["n_arrived"] == b["n_vehicles"]
    _compare(b, 1500, 0)


def test_truck_corridors():
    ty = np.array([1, 0], np.uint8)
    b = corridor(length=30000, departs=(0.0, 12.0), v0_mult=np.array([0.8, 1.0]), params=TRUCKS)
    _compare(dict(b, veh_type=ty), 1500, 1)
    _compare(dict(b, veh_type=ty[::-1].copy()), 1500, 1)
    # platoons of mixed types over a lane drop, ragged edge lengths
    rng = np.random.default_rng(1)
    for length in (61, 129, 300):
        b = corridor(n_edges=5, length=length, lanes=3, vlim=13.0, departs=np.arange(60) * 1.5, params=TRUCKS)
        _compare(dict(b, veh_type=(rng.random(60) < 0.4).astype(np.uint8)), 900, 1)


def test_amber_and_movement_phases_on_chains():
    sig = (np.full(7, 20), np.full(7, 4), np.arange(7) * 5)
    for ctrl in (W.CTRL_SIGNAL, W.CTRL_SIGNAL_NM):
        for amber in (0, 6):
            b = corridor(n_edges=6, length=300, departs=np.arange(40) * 3.0, ctrl=ctrl, sig=sig, steps=1500,
                         params=dict(amber_steps=amber))
            _compare(b, 1500, 1)


@pytest.mark.parametrize("name", ["cfg2_trucks", "cfg2_controls", "cfg2_trucks_controls"])
def test_config2_variants_prefix(name):
    b = W.by_name(name)
    _compare(b, 5000, 1, chunk=2500)


def test_validation_of_the_new_inputs(cfg1):
    import paper_1807_01148_b200 as pkg
    bad = [
        dict(cfg1, params=dict(cfg1["params"], n_types=5)),
        dict(cfg1, params=dict(cfg1["params"], n_types=2, type_len=(5, 1, 0, 0), type_a=(1, 1, 0, 0), type_vmax=(9, 9, 0, 0))),
        dict(cfg1, veh_type=np.full(cfg1["n_vehicles"], 1, np.uint8)),                       # type 1 without types
        dict(cfg1, node_ctrl=np.full(cfg1["n_nodes"], 5, np.uint8)),
        corridor(vlim=29.0, params=dict(lookahead_cells=16)),                                # shorter than a step + a vehicle
        dict(cfg1, params=dict(cfg1["params"], lookback_cells=0)),
        dict(W.with_controls(cfg1), params=dict(W.with_controls(cfg1)["params"], n_types=1, type_len=(15.5, 0, 0, 0),
                                                type_a=(1, 0, 0, 0), type_vmax=(99, 0, 0, 0), entry_zone_cells=40)),
    ]
    for n, b in enumerate(bad):
        with pytest.raises(pkg.TsError) as e:
            pkg.Sim(b, "cuda:0")
            pytest.fail(f"case {n} was accepted")
        assert e.value.code == pkg.binding.TS_EINVAL


def test_multi_step_digests_with_many_slots_per_thread():
    """ts_step_digest(n > 1) read counters that CTAs already in the next step were
    bumping.  Many slots per thread (64-thread CTAs, ~1e5 active vehicles), digests of 200 steps per
    call, against the oracle."""
    import paper_1807_01148_b200 as pkg
    from oracle import Oracle
    b = W.by_name("cfg3_dense")
    orc = Oracle(b)
    orc.set_threads(4)
    sim = pkg.Sim(b, "cuda:0")
    sim.set_option("threads", 64)
    for _ in range(3):
        want = orc.step(200, digests=True)
        got = sim.step_digest(200)
        bad = np.nonzero(want != got)[0]
        assert bad.size == 0, f"first digest mismatch at step {int(bad[0]) + 1} of the call"
    assert sim.read_counts()["n_active"] > 9472 * 10          # more than 10 slots per thread
    sim.close()


def test_utilisation_and_sampled_speed(cfg1):
    """ts_read_utilisation against the oracle's fp64 arithmetic on the same
    integer samples (fp32 on the device: 1e-6 relative), and its reset semantics."""
    import paper_1807_01148_b200 as pkg
    from oracle import Oracle, utilisation
    b = small_signal_grid()
    orc, sim = Oracle(b), pkg.Sim(b, "cuda:0")
    orc.step(1300); sim.step(1300)
    u, v = sim.read_utilisation()
    wu, wv = utilisation(orc.read_edge_stats(), b)
    assert wu.max() > 0.05
    assert np.allclose(u, wu, rtol=2e-6, atol=1e-9) and np.allclose(v, wv, rtol=2e-6, atol=1e-9)
    sim.read_edge_stats(reset=True)
    u, v = sim.read_utilisation()
    assert not u.any() and not v.any()
    sim.close()


def test_renumbered_edges_morton_order():
    """workload.renumber_edges / spatial_edge_order: the same network with its edges numbered along a
    space-filling curve is a different input (ties by edge index fall differently) and must match the
    oracle run on THAT input, bit for bit."""
    b = W.by_name("cfg4_small_morton")
    assert b["name"] == "cfg4_small_morton"
    _compare(b, 7200, 1, chunk=3600)


def test_both_code_plane_layouts(monkeypatch):
    """The code plane holds one byte per 4-cell granule where no two vehicles of a lane can come within
    4 cells of each other (every vehicle at least 4 m long, insert_clear_cells >= 4), else one byte per cell
    (DESIGN.md section 4).  Same results either way: the per-cell layout forced through the environment on
    the signal grid with trucks, and short vehicles (2.5 m, standing 3 m apart) that select it themselves."""
    b = W.with_trucks(small_signal_grid(), share=0.3)
    monkeypatch.setenv("TS_CODE_GRANULE", "0")
    _compare(b, b["steps"], 1)
    _compare(b, 600, 0)
    monkeypatch.delenv("TS_CODE_GRANULE")
    g = small_signal_grid()
    short = dict(g, params=dict(g["params"], veh_len=2.5, s0=0.5, insert_clear_cells=3))
    _compare(short, short["steps"], 1)
    tight = dict(g, params=dict(g["params"], veh_len=4.0, s0=0.25, insert_clear_cells=4))   # granule layout, queues 4 cells apart
    _compare(tight, tight["steps"], 1)
