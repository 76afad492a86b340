"""Parity of the CUDA path (through the C ABI) against the oracle, element by element.

Bar (BASELINE.json north_star): bit-exact on integer state and on the fp32 bit patterns of x
and v, at every step (64-bit digests) and in the final ts_read_state / ts_read_edge_stats.
"""
import numpy as np
import pytest

from test_oracle_invariants import small_signal_grid
from test_oracle_pins import corridor

pytestmark = pytest.mark.gpu


def _compare(bundle, steps, mode, chunk=None, **options):
    import paper_1807_01148_b200 as pkg
    from oracle import Oracle
    orc = Oracle(bundle)
    sim = pkg.Sim(bundle, "cuda:0", mode=mode)
    for key, value in options.items():
        sim.set_option(key, value)
    done = 0
    chunk = chunk or steps
    while done < steps:
        n = min(chunk, steps - done)
        want = orc.step(n, digests=True)
        got = sim.step_digest(n)
        bad = np.nonzero(want != got)[0]
        assert bad.size == 0, f"{bundle['name']}: first digest mismatch at step {done + int(bad[0]) + 1}"
        done += n
        if bundle["params"].get("emissions"):          # section 6.3.4 totals: fp32 bit patterns
            ma, mb = orc.read_emissions(), sim.read_emissions()
            for key in ("co_g", "fuel_ml"):
                assert (ma[key].view(np.uint32) == mb[key].view(np.uint32)).all(), f"{key} after step {done}"
    a, b = orc.read_state(), sim.read_state()
    for key in ("status", "edge", "lane", "cell", "route_idx", "insert_step", "arrive_step"):
        assert (a[key] == b[key]).all(), key
    for key in ("x", "v"):
        assert (a[key].view(np.uint32) == b[key].view(np.uint32)).all(), key
    for key in ("step", "n_pending", "n_active", "n_arrived"):
        assert a[key] == b[key], key
    assert b["vehicle_updates"] == orc.counters()["updates"]
    ea, eb = orc.read_edge_stats(), sim.read_edge_stats()
    for key in ea:
        assert np.array_equal(ea[key], eb[key]), key
    sim.close()
    return b


@pytest.mark.parametrize("mode", [1, 0])
def test_config1_full(cfg1, mode):
    st = _compare(cfg1, cfg1["steps"], mode, chunk=1000)
    assert st["n_arrived"] == 500


@pytest.mark.parametrize("mode", [1, 0])
def test_mixed_controls(mode):
    b = small_signal_grid()
    _compare(b, b["steps"], mode)


@pytest.mark.parametrize("options", [
    dict(sort_period=0),                       # never compacted: slots only grow
    dict(sort_period=1),                       # compacted + re-sorted after every step
    dict(sort_period=7, threads=128),          # several slots per thread, ragged tile tails
    dict(sort_period=50, threads=512, blocks_per_sm=2),
    dict(sort_period=3, threads=64),           # move records overflow shared memory into global
    dict(adaptive_chunk=37, adaptive_above=0),     # adaptive CTA size: the big size (768 threads) from the second chunk on
    dict(adaptive_chunk=50, adaptive_above=700),   # ... switching both ways as the slot count crosses 700
    dict(adaptive_chunk=1, adaptive_above=300, sort_period=5),
    dict(smem_tiles=0, threads=64, sort_period=16),    # every move record through L2
    dict(smem_tiles=1, threads=96, sort_groups=1),     # one tile in shared memory; re-sort by edge alone
    dict(sort_groups=2, sort_period=9),
])
def test_results_do_not_depend_on_slot_order(options):
    """A9/A10: compaction and the edge re-sort change where a vehicle's state lives, never what
    it is; neither does the launch geometry."""
    b = small_signal_grid()
    _compare(b, b["steps"], 1, **options)
    if options.get("sort_period") in (0, 1):
        _compare(b, 400, 0, sort_period=options["sort_period"])


def test_corridors():
    _compare(corridor(length=30000, vlim=29.0), 300, 1)
    _compare(corridor(length=30000, departs=(0.0, 10.0), v0_mult=np.array([0.8, 1.0])), 800, 1)
    N = 3
    sig = (np.full(N, 1), np.full(N, 60000), np.full(N, 1))
    _compare(corridor(n_edges=2, length=600, departs=np.arange(6) * 4.0, ctrl=2, sig=sig), 1200, 1)
    # ragged tails: edge lengths that are not multiples of 16, shortest legal edge
    for length in (16, 17, 31, 33, 47, 129):
        _compare(corridor(n_edges=5, length=length, lanes=2, vlim=13.0, departs=np.arange(30) * 1.5,
                          params=dict(entry_zone_cells=12)), 600, 1)


def test_config2_prefix():
    from paper_1807_01148_b200 import workload
    b = workload.config2()
    _compare(b, 4000, 1, chunk=2000)


def test_reset_reproduces(cfg1):
    import paper_1807_01148_b200 as pkg
    sim = pkg.Sim(cfg1, "cuda:0")
    a = sim.step_digest(900)
    sim.reset()
    b = sim.step_digest(900)
    assert (a == b).all()
    sim.reset()
    sim.step(900)                      # no digests: the plain timed path gives the same state
    sim2 = pkg.Sim(cfg1, "cuda:0")
    sim2.step_digest(900)
    s1, s2 = sim.read_state(), sim2.read_state()
    assert (s1["x"].view(np.uint32) == s2["x"].view(np.uint32)).all() and (s1["edge"] == s2["edge"]).all()


def test_empty_and_errors(cfg1):
    import paper_1807_01148_b200 as pkg
    sim = pkg.Sim(cfg1, "cuda:0")
    sim.step(0)
    st = sim.read_state()
    assert st["step"] == 0 and st["n_pending"] == 500 and (st["status"] == 0).all()
    bad = dict(cfg1); bad["edge_lanes"] = cfg1["edge_lanes"].copy(); bad["edge_lanes"][3] = 9
    with pytest.raises(pkg.TsError) as ei:
        pkg.Sim(bad, "cuda:0")
    assert ei.value.code == -1
    bad = dict(cfg1); bad["params"] = dict(cfg1["params"], entry_zone_cells=8)
    with pytest.raises(pkg.TsError):
        pkg.Sim(bad, "cuda:0")


@pytest.mark.parametrize("params", [
    dict(lookahead_cells=256, lookback_cells=256),      # scans longer than one 256-cell window
    dict(lookahead_cells=64, lookback_cells=32),
    dict(lc_period=3),                                  # stagger is a modulo, not a mask; one sort group
    dict(lc_period=0),                                  # lane changes off (P5)
    dict(lc_period=1),                                  # everybody evaluates every step
    dict(sample_period_steps=1),
    dict(sample_period_steps=0, insert_clear_cells=16),
    dict(dt=0.25, a=2.0, b=3.0, T=1.0, s0=1.0, veh_len=4.0, politeness=0.5, lc_threshold=0.2, b_safe=3.0),
])
def test_parameter_variants(params):
    """Every ts_params field away from its default, against the oracle with the same values."""
    b = small_signal_grid(seed=11, n_vehicles=900, steps=900)
    b = dict(b, params=dict(b["params"], **params))
    _compare(b, 900, 1)


def test_degenerate_inputs():
    import paper_1807_01148_b200 as pkg
    from paper_1807_01148_b200 import workload as W
    # no vehicles at all: steps run, nothing happens
    empty = corridor(departs=())
    sim = pkg.Sim(empty, "cuda:0")
    sim.step(50)
    st = sim.read_state()
    assert st["step"] == 50 and st["n_active"] == 0 and st["vehicle_updates"] == 0 and len(st["x"]) == 0
    assert sim.read_edge_stats()["n_samples"] == 0
    sim.close()
    # one-edge routes (arrive on the edge they start on), 8 lanes, the shortest and a very long edge
    _compare(corridor(n_edges=3, length=16, lanes=8, vlim=9.0, departs=np.arange(40) * 1.0, route_len=1,
                      params=dict(entry_zone_cells=12)), 300, 1)
    _compare(corridor(n_edges=1, length=65535, lanes=3, vlim=29.0, departs=np.arange(200) * 0.5), 1500, 1)
    # everybody wants the same cell at the same time: 300 vehicles, one origin edge, one departure time
    _compare(corridor(n_edges=4, length=120, lanes=2, vlim=13.0, departs=np.zeros(300), ctrl=W.CTRL_PRIORITY), 1200, 1)


def test_chunking_across_sort_boundaries():
    """ts_step(n) in uneven pieces: the host must know which slot set is current after every
    launch, whatever number of re-sorts fell inside it (sort period 7: launches of 1, 6, 7, 8, 13
    and 20 steps end just before, on and just after a boundary)."""
    import paper_1807_01148_b200 as pkg
    from oracle import Oracle
    b = small_signal_grid(seed=5, n_vehicles=700, steps=600)
    want = Oracle(b).step(600, digests=True)
    for mode in (1, 0):
        sim = pkg.Sim(b, "cuda:0", mode=mode)
        sim.set_option("sort_period", 7)
        got, pieces, i = [], (1, 6, 7, 8, 13, 20, 1, 1, 5), 0
        while len(got) < 600:
            n = min(pieces[i % len(pieces)], 600 - len(got))
            if i % 3 == 2:
                sim.step(n - 1) if n > 1 else None          # plain steps, then a digest for the last
                got.extend([None] * (n - 1))
                got.append(int(sim.step_digest(1)[0]))
            else:
                got.extend(int(d) for d in sim.step_digest(n))
            i += 1
        bad = [k for k, d in enumerate(got) if d is not None and d != int(want[k])]
        assert not bad, f"mode {mode}: first mismatch at step {bad[0] + 1}"
        st = sim.read_state()
        assert st["step"] == 600
        sim.close()


@pytest.mark.parametrize("seed", [11, 12, 13])
def test_signal_plans_of_every_shape(seed):
    """A1: the device reduces the signal test to one comparison after a modulo by multiplication.
    Plans that stress it: green of one step with no all-red (cycle = in-degree, down to 1),
    power-of-two and odd cycles, phases up to 65 535 steps, offsets up to 2^31 - 1."""
    rng = np.random.default_rng(seed)
    b = small_signal_grid(seed=seed, n_vehicles=900, steps=1200)
    N = b["n_nodes"]
    green = rng.choice([1, 2, 3, 7, 8, 16, 31, 64, 100, 257, 4096, 65535], N)
    allred = rng.choice([0, 0, 1, 2, 5, 8, 60], N)
    allred = np.where(green + allred > 65535, 0, allred)
    offset = rng.choice([0, 1, 5, 1000, 2 ** 24 + 3, 2 ** 31 - 1, 2 ** 31 - 2, 123456789], N)
    b = dict(b, sig_green_steps=green.astype(np.uint32), sig_allred_steps=allred.astype(np.uint32),
             sig_offset_steps=offset.astype(np.uint32))
    _compare(b, 1200, 1, chunk=400)
    _compare(b, 300, 0)
    if seed == 11:                             # one inbound edge, green 1 + all-red 0: cycle 1, always green
        n = 3
        one = (np.full(n, 1), np.full(n, 0), np.full(n, 2 ** 31 - 1))
        _compare(corridor(n_edges=2, length=300, departs=np.arange(8) * 3.0, ctrl=2, sig=one), 600, 1)
        two = (np.full(n, 1), np.full(n, 1), np.full(n, 7))            # cycle 2: green on alternate steps
        _compare(corridor(n_edges=2, length=300, departs=np.arange(8) * 3.0, ctrl=2, sig=two), 600, 1)


def test_checkpoint_and_resume_give_the_uninterrupted_run():
    """ts_checkpoint / ts_restore: stepping on from a restored checkpoint reproduces, digest by digest, what the
    uninterrupted run (and the oracle) give -- across a re-sort boundary, in the adaptive launch scheme, into a
    second simulation object created from the same inputs, and with a re-routed demand in the workspace."""
    import paper_1807_01148_b200 as pkg
    from oracle import Oracle
    from paper_1807_01148_b200 import workload as W
    b = small_signal_grid()
    b = dict(b, params=dict(b["params"], emissions=1, route_capacity=2 * len(b["route_edges"]) + 1024))
    want = Oracle(b).step(1500, digests=True)
    sim = pkg.Sim(b, "cuda:0")
    sim.set_option("adaptive_chunk", 64)
    assert np.array_equal(sim.step_digest(700), want[:700])
    snap = sim.checkpoint()
    assert np.array_equal(sim.step_digest(800), want[700:])                  # the uninterrupted run
    first = sim.read_state()
    sim.restore(snap)
    assert sim.read_counts()["step"] == 700
    assert np.array_equal(sim.step_digest(800), want[700:])                  # resumed in place
    again = sim.read_state()
    for key in ("status", "edge", "lane", "route_idx", "insert_step", "arrive_step"):
        assert np.array_equal(first[key], again[key]), key
    assert np.array_equal(first["x"].view(np.uint32), again["x"].view(np.uint32))
    ea, eb = sim.read_emissions(), None
    other = pkg.Sim(b, "cuda:0")                                             # a fresh object, same inputs
    other.restore(snap)
    assert np.array_equal(other.step_digest(800), want[700:])
    eb = other.read_emissions()
    assert np.array_equal(ea["fuel_ml"].view(np.uint32), eb["fuel_ml"].view(np.uint32))
    es1, es2 = sim.read_edge_stats(), other.read_edge_stats()
    for key in es1:
        assert np.array_equal(es1[key], es2[key]), key
    # a checkpoint taken after ts_reroute carries the new routes and queues
    wf = W.free_flow_weights(b)
    other.reroute(wf, W.reroute_mask(b["n_vehicles"], 2))
    off, edges = other.read_routes()
    snap2 = other.checkpoint()
    d1 = other.step_digest(600)
    other.reroute(wf)                                                        # something else in the workspace
    other.restore(snap2)
    o2, e2 = other.read_routes()
    assert np.array_equal(off, o2) and np.array_equal(edges, e2)
    assert np.array_equal(other.step_digest(600), d1)
    assert np.array_equal(d1, Oracle(dict(b, route_off=off, route_edges=edges)).step(600, digests=True))
    # refused: a checkpoint of other inputs, or no checkpoint at all
    small = pkg.Sim(W.config1(), "cuda:0")
    with pytest.raises(pkg.TsError):
        small.restore(snap)
    with pytest.raises(pkg.TsError):
        sim.restore(np.zeros(len(snap), np.uint8))
    for s_ in (sim, other, small):
        s_.close()
