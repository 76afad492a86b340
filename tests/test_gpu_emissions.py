"""Parity of the section 6.3.4 accumulators (CO, Eq. 8; fuel, Eq. 9; SURVEY.md
8(f) row 2) of the CUDA path against the oracle: fp32 bit patterns of every vehicle's totals.
The traffic digests are compared on the way, so these runs also show that switching the
accumulators on changes nothing else."""
import numpy as np
import pytest

from test_gpu_parity import _compare
from test_oracle_invariants import small_signal_grid
from test_oracle_pins import corridor

pytestmark = pytest.mark.gpu


def _with_emissions(b):
    return dict(b, params=dict(b["params"], emissions=1))


@pytest.mark.parametrize("mode", [1, 0])
def test_config1_full(cfg1, mode):
    _compare(_with_emissions(cfg1), cfg1["steps"], mode, chunk=900)


@pytest.mark.parametrize("options", [
    dict(sort_period=0), dict(sort_period=1), dict(sort_period=7, threads=128),
    dict(sort_period=50, threads=512, blocks_per_sm=2), dict(sort_period=3, threads=64),
    dict(adaptive_chunk=50, adaptive_above=700),
])
def test_totals_do_not_depend_on_slot_order(options):
    """The pair is indexed by vehicle id, so compaction, the re-sort and the launch geometry
    cannot change it."""
    b = _with_emissions(small_signal_grid())
    _compare(b, b["steps"], 1, chunk=257, **options)


def test_corridors_and_red_line():
    _compare(_with_emissions(corridor(length=30000, vlim=29.0)), 300, 1, chunk=100)
    N = 3
    sig = (np.full(N, 1), np.full(N, 60000), np.full(N, 1))
    _compare(_with_emissions(corridor(n_edges=2, length=600, departs=np.arange(6) * 4.0, ctrl=2, sig=sig)),
             1200, 1, chunk=400)


def test_config2_prefix():
    from paper_1807_01148_b200 import workload as W
    _compare(_with_emissions(W.by_name("cfg2")), 4000, 1, chunk=1000)


def test_full_size_config5_prefix():
    """BASELINE.json config 5 at full size (2 M vehicles), default launch configuration: the first
    2 400 steps (the whole 15-minute release and the spillback it causes), every vehicle's totals."""
    from paper_1807_01148_b200 import workload as W
    _compare(_with_emissions(W.by_name("cfg5")), 2400, 1, chunk=1200)


def test_reset_disabled_and_edge_stat_reset(cfg1):
    import paper_1807_01148_b200 as pkg
    from paper_1807_01148_b200 import binding
    sim = pkg.Sim(cfg1, "cuda:0")
    sim.step(10)
    with pytest.raises(binding.TsError) as ei:
        sim.read_emissions()
    assert ei.value.code == binding.TS_EINVAL
    sim.close()
    sim = pkg.Sim(_with_emissions(cfg1), "cuda:0")
    sim.step(600)
    first = sim.read_emissions()
    assert first["co_g"].sum() > 0 and first["fuel_ml"].sum() > 0
    sim.read_edge_stats(reset=True)            # resets the edge statistics only
    again = sim.read_emissions()
    assert np.array_equal(first["co_g"], again["co_g"]) and np.array_equal(first["fuel_ml"], again["fuel_ml"])
    sim.reset()
    zero = sim.read_emissions()
    assert not zero["co_g"].any() and not zero["fuel_ml"].any()
    sim.step(600)
    second = sim.read_emissions()
    assert np.array_equal(first["co_g"], second["co_g"]) and np.array_equal(first["fuel_ml"], second["fuel_ml"])
    sim.close()
