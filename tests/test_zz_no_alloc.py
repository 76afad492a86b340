"""ts_sssp_static: the shortest-path tree kernel with its scratch in a static device array, for callers
that cannot allocate (include/trafficsim.h).  Its trees must give the SAME routes as the existing path
(ts_reroute, whose scratch is carved from the caller's workspace) from the same weights -- integer work,
so the comparison is exact, like every routing test here -- on two calls in a row that share the array
(the second sees the first one's leftovers), then on a graph of another size, and sizes beyond the stated
maximum must be refused.  Collected last on purpose (pytest -x): a failure here hides no other test."""
import numpy as np
import pytest

from paper_1807_01148_b200 import workload as W

pytestmark = pytest.mark.gpu


def _csr(b):
    """Outbound edges by tail node, edge ids ascending inside a node."""
    ef = b["edge_from"].astype(np.int64)
    order = np.argsort(ef, kind="stable")
    off = np.zeros(b["n_nodes"] + 1, np.int64)
    np.add.at(off, ef + 1, 1)
    return np.cumsum(off).astype(np.int32), order.astype(np.int32)


def _routes_from_trees(b, pred, sources):
    """Every vehicle's route read off the trees: walk back from its destination to its origin."""
    ef, et = b["edge_from"].astype(np.int64), b["edge_to"].astype(np.int64)
    off, re = b["route_off"].astype(np.int64), b["route_edges"].astype(np.int64)
    origin, dest = ef[re[off[:-1]]], et[re[off[1:] - 1]]
    row = np.searchsorted(sources, origin)
    assert (sources[row] == origin).all()
    V = len(origin)
    cur, steps = dest.copy(), []
    live = cur != origin
    while live.any():
        e = np.where(live, pred[row, cur].astype(np.int64), -1)
        assert (e[live] != 0xFFFFFFFF).all(), "a destination the tree does not reach"
        steps.append(e)
        cur = np.where(live, ef[np.maximum(e, 0)], cur)
        live = cur != origin
        assert len(steps) <= b["n_nodes"]
    walked = np.stack(steps, 1)                               # [V, longest], destination first, -1 = done
    length = (walked >= 0).sum(1)
    new_off = np.zeros(V + 1, np.int64)
    new_off[1:] = np.cumsum(length)
    out = np.zeros(int(new_off[-1]), np.int64)
    i, j = np.nonzero(walked >= 0)
    out[new_off[i] + length[i] - 1 - j] = walked[i, j]
    return new_off.astype(np.uint64), out.astype(np.uint32)


class _Graph:
    """The caller's device buffers: allocated ONCE, before any call of the entry point."""

    def __init__(self, b, torch):
        dev = "cuda:0"
        off, order = _csr(b)
        ef, re, ro = b["edge_from"].astype(np.int64), b["route_edges"].astype(np.int64), b["route_off"].astype(np.int64)
        self.b, self.N = b, b["n_nodes"]
        self.sources = np.unique(ef[re[ro[:-1]]])
        t = lambda a: torch.from_numpy(np.ascontiguousarray(a, np.int32)).to(dev)
        self.out_off, self.out_edge = t(off), t(order)
        self.edge_to, self.src = t(b["edge_to"].astype(np.int32)), t(self.sources.astype(np.int32))
        self.w = [torch.zeros(b["n_edges"], dtype=torch.int32, device=dev) for _ in range(2)]
        self.pred = [torch.zeros(len(self.sources) * self.N, dtype=torch.int32, device=dev) for _ in range(2)]
        self.err = torch.zeros(1, dtype=torch.int32, device=dev)

    def call(self, pkg, slot):
        pkg.sssp_static(self.N, self.out_off, self.out_edge, self.edge_to, self.w[slot], self.src, self.pred[slot], self.err)

    def trees(self, slot):
        return self.pred[slot].cpu().numpy().view(np.uint32).reshape(len(self.sources), self.N)


def _existing_path(pkg, b, steps_before):
    """Weights and routes of ts_reroute after `steps_before` simulated steps, twice in a row."""
    cap = 2 * len(b["route_edges"]) + 1024
    sim = pkg.Sim(dict(b, params=dict(b["params"], route_capacity=cap)), "cuda:0")
    wf = W.free_flow_weights(b)
    out = []
    for n in steps_before:
        if n:
            sim.step(n)
        info = sim.reroute(wf)
        out.append((info["w"].copy(), sim.read_routes()))
    sim.close()
    return out


def test_static_scratch_trees_give_the_routes_of_the_existing_path():
    import torch
    import paper_1807_01148_b200 as pkg
    b = W.config2()
    (w1, routes1), (w2, routes2) = _existing_path(pkg, b, (3000, 2500))
    assert not np.array_equal(w1, w2)                          # two different problems
    g = _Graph(b, torch)
    small = W.config1()
    (w3, routes3), = _existing_path(pkg, small, (1200,))
    gs = _Graph(small, torch)
    for slot, w in ((0, w1), (1, w2)):
        g.w[slot].copy_(torch.from_numpy(w.astype(np.int32)))
    gs.w[0].copy_(torch.from_numpy(w3.astype(np.int32)))
    torch.cuda.synchronize()

    g.call(pkg, 0)                                             # first call: resolves the array's address
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]
    g.call(pkg, 1)                                             # two calls in a row on the shared array ...
    g.call(pkg, 0)                                             # ... the first problem again over the second's leftovers
    gs.call(pkg, 0)                                            # ... and a graph of another size over both
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] >= free_before         # the calls took no device memory

    for slot, (want_off, want_edges) in ((0, routes1), (1, routes2)):
        got_off, got_edges = _routes_from_trees(b, g.trees(slot), g.sources)
        assert np.array_equal(got_off, want_off), f"call {slot}: route offsets"
        assert np.array_equal(got_edges, want_edges), f"call {slot}: route edges"
    got_off, got_edges = _routes_from_trees(small, gs.trees(0), gs.sources)
    assert np.array_equal(got_off, routes3[0]) and np.array_equal(got_edges, routes3[1])
    assert int(g.err.item()) == 0 and int(gs.err.item()) == 0


def test_sizes_beyond_the_static_maximum_are_refused():
    import torch
    import paper_1807_01148_b200 as pkg
    limit = int(pkg.load().ts_sssp_static_max_nodes())
    assert limit == 65536
    z = torch.zeros(8, dtype=torch.int32, device="cuda:0")
    with pytest.raises(pkg.TsError) as e:
        pkg.sssp_static(limit + 1, z, z, z, z, z, z)
    assert e.value.code == pkg.binding.TS_EINVAL and "exceed" in str(e.value) and str(limit) in str(e.value)
    pkg.sssp_static(4, z, z, z, z, z[:0], z)                   # no sources: nothing to do, nothing launched
