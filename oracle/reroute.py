"""ORACLE -- test infrastructure, not product code.

Iterative decaying re-routing, PAPER.md:386 (section 6.3.1) and PAPER.md:431 (section 6.3.5):
"In the first iteration, we use the initialization formula above to compute the edge weight for
routing.  After that first iteration, we use the microsimulation measurements to update those
weights and repeat the microsimulation ... we recompute all routes the first and second
iteration, and then we decay it to half and one-fourth of the vehicles", with shortest paths for
all vehicles at once ("we replace it with ... All Pairs Shortest Path").

Plain numpy; SciPy's Dijkstra is the one library step.  Readings (R37-R40):
  R37  edge weights are INTEGERS in units of 1/256 simulation step, so that path costs are exact and
       the chosen routes are a function of the inputs alone: measured weight of an edge that at
       least one vehicle left = round-half-up(256 * exit_steps_sum / exited), else the caller's
       free-flow weight w_free[e] (the paper's initialisation, an input); clamped to [1, 2^20].
  R38  a vehicle keeps its origin node (tail of its first edge) and destination node (head of its
       last edge); its new route is THE shortest path under these weights, made unique by taking,
       at every node on the way back from the destination, the inbound edge with the smallest
       (dist[tail] + w, edge id).
  R39  which vehicles are re-routed in an iteration is an input (a mask drawn by the caller from a
       seed: all, all, 1/2, 1/4 -- workload.reroute_mask); the others keep their route.
  R40  a vehicle whose origin equals its destination, or whose destination cannot be reached,
       keeps its route.
Only tests/ and bench.py's oracle legs may import this module; it imports nothing from the package.
"""
from __future__ import annotations

import numpy as np
import scipy.sparse as sp
from scipy.sparse.csgraph import dijkstra

W_UNIT = 256           # weight units per simulation step (R37)
W_MAX = 1 << 20


def edge_weights(exited, exit_steps_sum, w_free):
    """R37.  All integer arithmetic (Python ints via uint64 numpy)."""
    exited = np.asarray(exited, np.uint64)
    s = np.asarray(exit_steps_sum, np.uint64)
    w = np.asarray(w_free, np.uint64).copy()
    has = exited > 0
    w[has] = (s[has] * np.uint64(W_UNIT) + exited[has] // np.uint64(2)) // exited[has]
    return np.clip(w, 1, W_MAX).astype(np.uint32)


def shortest_path_trees(n_nodes, edge_from, edge_to, w, sources):
    """dist[s, v] (exact integers in float64; inf = unreachable) and pred_edge[s, v] by rule R38
    (-1 at the source and at unreachable nodes)."""
    ef = np.asarray(edge_from, np.int64); et = np.asarray(edge_to, np.int64)
    w = np.asarray(w, np.float64)
    E = len(ef)
    # parallel edges: the graph matrix keeps the cheapest one per (tail, head); ties and the edge
    # ids are settled below from dist, not from the matrix
    order = np.lexsort((w, et, ef))
    first = np.ones(E, bool)
    first[1:] = (ef[order][1:] != ef[order][:-1]) | (et[order][1:] != et[order][:-1])
    keep = order[first]
    g = sp.csr_matrix((w[keep], (ef[keep], et[keep])), shape=(n_nodes, n_nodes))
    dist = np.atleast_2d(dijkstra(g, directed=True, indices=np.asarray(sources, np.int64)))
    pred = np.full(dist.shape, -1, np.int64)
    for r in range(dist.shape[0]):
        d = dist[r]
        cand = d[ef] + w                                   # cost of reaching head(e) through e
        tight = np.isfinite(cand) & (cand == d[et]) & (et != sources[r])
        e_ids = np.nonzero(tight)[0]                       # ascending edge id
        # the smallest edge id among the tight inbound edges of each node
        heads, idx = np.unique(et[e_ids], return_index=True)
        pred[r, heads] = e_ids[idx]
    return dist, pred


def reroute(bundle, exited, exit_steps_sum, w_free, mask=None):
    """New (route_off, route_edges, w) for the bundle's vehicles (R37-R40)."""
    b = bundle
    N = int(b["n_nodes"])
    ef = np.asarray(b["edge_from"], np.int64); et = np.asarray(b["edge_to"], np.int64)
    off = np.asarray(b["route_off"], np.int64); re = np.asarray(b["route_edges"], np.int64)
    V = int(b["n_vehicles"])
    mask = np.ones(V, bool) if mask is None else np.asarray(mask, bool)
    w = edge_weights(exited, exit_steps_sum, w_free)
    origin = ef[re[off[:-1]]]
    dest = et[re[off[1:] - 1]]
    sources = np.unique(origin[mask]) if mask.any() else np.zeros(0, np.int64)
    routes = [re[off[i]:off[i + 1]] for i in range(V)]
    batch = 64
    for lo in range(0, len(sources), batch):
        src = sources[lo:lo + batch]
        dist, pred = shortest_path_trees(N, ef, et, w, src)
        row_of = {int(s): r for r, s in enumerate(src)}
        todo = np.nonzero(mask & np.isin(origin, src))[0]
        for i in todo:
            r = row_of[int(origin[i])]
            o, d = int(origin[i]), int(dest[i])
            if o == d or not np.isfinite(dist[r, d]):
                continue                                    # R40
            path = []
            v = d
            while v != o:
                e = int(pred[r, v])
                path.append(e)
                v = int(ef[e])
            routes[i] = np.asarray(path[::-1], np.int64)
    new_off = np.zeros(V + 1, np.uint64)
    new_off[1:] = np.cumsum([len(p) for p in routes])
    new_edges = np.concatenate(routes).astype(np.uint32) if V else np.zeros(0, np.uint32)
    return new_off, new_edges, w
