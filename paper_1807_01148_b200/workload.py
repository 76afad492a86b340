"""Seeded synthetic workloads.

This module serves BOTH the oracle and the CUDA path and therefore holds none of the
method's arithmetic: it builds road networks, traffic controls, origin/destination pairs,
free-flow shortest-path routes and departure times, and nothing else.  The inputs stand in
for the paper's OpenStreetMap Bay Area network and ActivitySim demand
(PAPER.md:148, :366), neither of which exists in this container.

A *bundle* is a plain dict of NumPy arrays with exactly the fields of the C ABI
(include/trafficsim.h): network (edge_from, edge_to, edge_len_m, edge_lanes, edge_vlim,
node_ctrl, sig_*), routes (route_off, route_edges), departures (depart_time_s, v0_mult,
mand_dist_m), `params` (dict) and `steps`.
"""
from __future__ import annotations

import hashlib
import multiprocessing as mp
import os

import numpy as np
import scipy.sparse as sp
from scipy.sparse.csgraph import connected_components, dijkstra

SEED_BASE = 180701148  # arxiv id; config n uses SEED_BASE + n (SURVEY.md:476)

CTRL_FREE, CTRL_PRIORITY, CTRL_SIGNAL = 0, 1, 2
CTRL_STOP, CTRL_SIGNAL_NM = 3, 4     # control variants of PAPER.md:402 (readings R34, R35)

# A second vehicle type "to represent trucks ... size, acceleration, and maximum speed".
# The paper prints no values; these are this repository's (reading R31): type 0 = car with
# the BASELINE.json config 1 values, type 1 = truck, 12 m long, half the acceleration, 25 m/s cap.
TRUCK_PARAMS = dict(n_types=2, type_len=(5.0, 12.0, 0.0, 0.0), type_a=(1.0, 0.5, 0.0, 0.0),
                    type_vmax=(1000.0, 25.0, 0.0, 0.0), insert_clear_cells=14)

DEFAULT_PARAMS = dict(
    dt=0.5, a=1.0, b=1.5, T=1.5, s0=2.0, veh_len=5.0,            # BASELINE.json config 1
    b_safe=4.0, politeness=0.2, lc_threshold=0.1,                # BASELINE.json config 2
    mand_dist_default=100.0,
    lookahead_cells=128, lookback_cells=128, lc_period=4, entry_zone_cells=32,
    insert_clear_cells=7, sample_period_steps=120,               # PAPER.md:437 one minute
)


# --------------------------------------------------------------------------- bundle helpers

def make_bundle(name, n_nodes, edge_from, edge_to, edge_len_m, edge_lanes, edge_vlim,
                node_ctrl, route_off, route_edges, depart_time_s, steps,
                sig_green_steps=None, sig_allred_steps=None, sig_offset_steps=None,
                v0_mult=None, mand_dist_m=None, params=None, node_xy=None, veh_type=None):
    """Normalise dtypes and fill defaults.  Used by the generators and by hand-made tests."""
    n_nodes = int(n_nodes)
    z = np.zeros(n_nodes, np.uint32)
    prm = dict(DEFAULT_PARAMS)
    prm.update(params or {})
    V = len(depart_time_s)
    b = dict(
        name=name, n_nodes=n_nodes, n_edges=int(len(edge_from)), n_vehicles=int(V),
        edge_from=np.ascontiguousarray(edge_from, np.uint32),
        edge_to=np.ascontiguousarray(edge_to, np.uint32),
        edge_len_m=np.ascontiguousarray(edge_len_m, np.uint32),
        edge_lanes=np.ascontiguousarray(edge_lanes, np.uint8),
        edge_vlim=np.ascontiguousarray(edge_vlim, np.float32),
        node_ctrl=np.ascontiguousarray(node_ctrl, np.uint8),
        sig_green_steps=np.ascontiguousarray(z if sig_green_steps is None else sig_green_steps, np.uint32),
        sig_allred_steps=np.ascontiguousarray(z if sig_allred_steps is None else sig_allred_steps, np.uint32),
        sig_offset_steps=np.ascontiguousarray(z if sig_offset_steps is None else sig_offset_steps, np.uint32),
        route_off=np.ascontiguousarray(route_off, np.uint64),
        route_edges=np.ascontiguousarray(route_edges, np.uint32),
        depart_time_s=np.ascontiguousarray(depart_time_s, np.float32),
        v0_mult=np.ascontiguousarray(np.ones(V) if v0_mult is None else v0_mult, np.float32),
        mand_dist_m=np.ascontiguousarray(
            np.full(V, prm["mand_dist_default"]) if mand_dist_m is None else mand_dist_m, np.float32),
        params=prm, steps=int(steps),
    )
    if node_xy is not None:
        b["node_xy"] = np.asarray(node_xy, np.float64)
    if veh_type is not None:
        b["veh_type"] = np.ascontiguousarray(veh_type, np.uint8)
    return b


_HASH_FIELDS = ("edge_from", "edge_to", "edge_len_m", "edge_lanes", "edge_vlim", "node_ctrl",
                "sig_green_steps", "sig_allred_steps", "sig_offset_steps", "route_off",
                "route_edges", "depart_time_s", "v0_mult", "mand_dist_m")


def bundle_sha256(b) -> str:
    """Checksum of every array the simulators read: detects generator drift between machines."""
    h = hashlib.sha256()
    for f in _HASH_FIELDS:
        h.update(f.encode())
        h.update(np.ascontiguousarray(b[f]).tobytes())
    if b.get("veh_type") is not None:
        h.update(b"veh_type")
        h.update(np.ascontiguousarray(b["veh_type"]).tobytes())
    h.update(repr(sorted(b["params"].items())).encode())
    return h.hexdigest()


def draw_mand_dist(rng, V, D=100.0):
    """Reading R11: P(mandatory at distance x from the exit) = exp(-(x/D)^2),
    realised as a per-vehicle threshold drawn on the host, D*sqrt(-ln u), u ~ U(0,1)."""
    u = rng.random(V)
    u = np.clip(u, 1e-12, 1.0)
    return (D * np.sqrt(-np.log(u))).astype(np.float32)


# --------------------------------------------------------------------------- routing

_G = {}  # graph shared with forked workers


def _route_batch(args):
    """Free-flow shortest paths for all vehicles of a batch of origin nodes."""
    origins, veh_lists = args
    csr, in_from, in_eid, dests = _G["csr"], _G["in_from"], _G["in_eid"], _G["dests"]
    _, pred = dijkstra(csr, directed=True, indices=origins, return_predecessors=True)
    pred = np.atleast_2d(pred)
    veh = np.concatenate(veh_lists)
    row = np.concatenate([np.full(len(v), i, np.int64) for i, v in enumerate(veh_lists)])
    cur = dests[veh].astype(np.int64)
    org = np.asarray(origins, np.int64)[row]
    hops_v, hops_e = [], []
    alive = np.nonzero(cur != org)[0]
    while alive.size:
        c = cur[alive]
        p = pred[row[alive], c].astype(np.int64)
        if (p < 0).any():
            raise RuntimeError("destination unreachable: network not strongly connected")
        cand = in_from[c]                                 # [n, maxdeg]
        slot = np.argmax(cand == p[:, None], axis=1)      # first match = cheapest in-edge
        hops_v.append(alive)
        hops_e.append(in_eid[c, slot])
        cur[alive] = p
        alive = alive[p != org[alive]]
    n = len(veh)
    length = np.zeros(n, np.int64)
    for a in hops_v:
        length[a] += 1
    off = np.zeros(n + 1, np.int64)
    np.cumsum(length, out=off[1:])
    edges = np.empty(off[-1], np.uint32)
    fill = off[1:].copy()                                  # fill each route from its end
    for a, e in zip(hops_v, hops_e):
        fill[a] -= 1
        edges[fill[a]] = e
    return veh, length, edges


def shortest_path_routes(n_nodes, edge_from, edge_to, weight, origins, dests, workers=None,
                         batch=None):
    """route_off/route_edges for every (origin, dest) pair by Dijkstra on `weight`
    (free-flow time, Eq. 4; BASELINE.json 'routes = CPU shortest path')."""
    E = len(edge_from)
    V = len(origins)
    order = np.lexsort((np.arange(E), weight, edge_to))    # in-edges per node, cheapest first
    indeg = np.bincount(edge_to, minlength=n_nodes)
    maxdeg = int(indeg.max())
    start = np.zeros(n_nodes + 1, np.int64)
    np.cumsum(indeg, out=start[1:])
    slot = np.arange(E) - start[edge_to[order]]
    in_from = np.full((n_nodes, maxdeg), -1, np.int64)
    in_eid = np.zeros((n_nodes, maxdeg), np.uint32)
    in_from[edge_to[order], slot] = edge_from[order]
    in_eid[edge_to[order], slot] = order
    # parallel edges: keep the cheapest in the matrix (csr would sum duplicates)
    key = edge_from.astype(np.int64) * n_nodes + edge_to
    o2 = np.lexsort((weight, key))
    first = np.ones(E, bool)
    first[1:] = key[o2][1:] != key[o2][:-1]
    keep = o2[first]
    csr = sp.csr_matrix((weight[keep].astype(np.float64), (edge_from[keep], edge_to[keep])),
                        shape=(n_nodes, n_nodes))
    _G.update(csr=csr, in_from=in_from, in_eid=in_eid, dests=np.asarray(dests, np.int64))

    origins = np.asarray(origins, np.int64)
    vorder = np.argsort(origins, kind="stable")
    uniq, ustart = np.unique(origins[vorder], return_index=True)
    uend = np.append(ustart[1:], V)
    if batch is None:
        batch = max(1, min(64, (32 << 20) // max(1, 4 * n_nodes)))
    tasks = []
    for i in range(0, len(uniq), batch):
        tasks.append((uniq[i:i + batch],
                      [vorder[ustart[j]:uend[j]] for j in range(i, min(i + batch, len(uniq)))]))
    workers = workers or min(len(tasks), os.cpu_count() or 1)
    if workers > 1 and len(tasks) > 1:
        with mp.get_context("fork").Pool(workers) as pool:
            results = pool.map(_route_batch, tasks, chunksize=1)
    else:
        results = [_route_batch(t) for t in tasks]
    length = np.zeros(V, np.int64)
    for veh, ln, _ in results:
        length[veh] = ln
    route_off = np.zeros(V + 1, np.uint64)
    np.cumsum(length, out=route_off[1:])
    route_edges = np.empty(int(route_off[-1]), np.uint32)
    for veh, ln, edges in results:
        src_off = np.zeros(len(veh) + 1, np.int64)
        np.cumsum(ln, out=src_off[1:])
        # scatter each vehicle's slice; vectorised via repeat
        dst = np.repeat(route_off[veh].astype(np.int64) - src_off[:-1], ln) + np.arange(src_off[-1])
        route_edges[dst] = edges
    _G.clear()
    return route_off, route_edges


# --------------------------------------------------------------------------- networks

def _grid_undirected(W, Hh):
    """4-neighbour grid: returns (u, v) node pairs, row-major node ids."""
    idx = np.arange(W * Hh).reshape(Hh, W)
    horiz = np.stack([idx[:, :-1].ravel(), idx[:, 1:].ravel()], 1)
    vert = np.stack([idx[:-1, :].ravel(), idx[1:, :].ravel()], 1)
    return np.concatenate([horiz, vert], 0)


def _directed(und, *attrs):
    """Both directions of every undirected edge, sharing its attributes."""
    ef = np.concatenate([und[:, 0], und[:, 1]])
    et = np.concatenate([und[:, 1], und[:, 0]])
    return (ef, et) + tuple(np.concatenate([a, a]) for a in attrs)


def _largest_scc(n_nodes, ef, et):
    g = sp.csr_matrix((np.ones(len(ef)), (ef, et)), shape=(n_nodes, n_nodes))
    _, lab = connected_components(g, directed=True, connection="strong")
    big = np.argmax(np.bincount(lab))
    keep_node = lab == big
    remap = np.full(n_nodes, -1, np.int64)
    remap[keep_node] = np.arange(keep_node.sum())
    keep_edge = keep_node[ef] & keep_node[et]
    return keep_node, remap, keep_edge


def _signal_arrays(rng, n_nodes, et, signal_nodes, green, allred):
    """Per-node green/all-red (steps) and a uniform offset within the node's cycle."""
    n_in = np.bincount(et, minlength=n_nodes)
    g = np.zeros(n_nodes, np.uint32)
    r = np.zeros(n_nodes, np.uint32)
    o = np.zeros(n_nodes, np.uint32)
    g[signal_nodes] = np.broadcast_to(green, n_nodes)[signal_nodes] if np.ndim(green) else green
    r[signal_nodes] = allred
    cyc = np.maximum(1, n_in * (g.astype(np.int64) + r))
    o[signal_nodes] = (rng.random(n_nodes) * cyc).astype(np.uint32)[signal_nodes]
    return g, r, o


def _gravity_dests(rng, xy, origins_unique, counts, scale_m):
    """Destination node for each trip: P(dest | origin) ~ exp(-d/scale), Euclidean d, dest != origin."""
    out = []
    for o, cnt in zip(origins_unique, counts):
        d = np.hypot(xy[:, 0] - xy[o, 0], xy[:, 1] - xy[o, 1])
        w = np.exp(-d / scale_m)
        w[o] = 0.0
        cdf = np.cumsum(w)
        out.append(np.searchsorted(cdf, rng.random(cnt) * cdf[-1], side="right"))
    return np.minimum(np.concatenate(out), len(xy) - 1)


def _finish(name, rng, n_nodes, ef, et, length, lanes, vlim, ctrl, sig, origins, dests,
            depart, steps, v0_mult, params, xy, workers):
    weight = length.astype(np.float64) / vlim.astype(np.float64)       # PAPER.md:224 Eq. 4
    route_off, route_edges = shortest_path_routes(n_nodes, ef, et, weight, origins, dests, workers)
    V = len(origins)
    return make_bundle(name, n_nodes, ef, et, length, lanes, vlim, ctrl, route_off, route_edges,
                       depart, steps, sig[0], sig[1], sig[2], v0_mult,
                       draw_mand_dist(rng, V), params, xy)


# --------------------------------------------------------------------------- the five configs

def config1(n_vehicles=500, steps=3600, grid=4, workers=1):
    """BASELINE.json configs[0] 'tiny': 4x4 grid, 200 m, 2 lanes, 15 m/s, PRIORITY junctions."""
    rng = np.random.default_rng(SEED_BASE + 1)
    N = grid * grid
    und = _grid_undirected(grid, grid)
    ef, et = _directed(und)
    E = len(ef)
    xy = np.stack([np.arange(N) % grid, np.arange(N) // grid], 1) * 200.0
    origins = rng.integers(0, N, n_vehicles)
    dests = (origins + rng.integers(1, N, n_vehicles)) % N
    depart = rng.random(n_vehicles) * 300.0
    z = np.zeros(N, np.uint32)
    return _finish("cfg1_tiny", rng, N, ef, et, np.full(E, 200), np.full(E, 2), np.full(E, 15.0),
                   np.full(N, CTRL_PRIORITY), (z, z, z), origins, dests, depart, steps,
                   np.ones(n_vehicles), None, xy, workers)


def config2(n_vehicles=20000, steps=14400, grid=32, workers=None):
    """configs[1]: 32x32 grid, lengths U(100,400), 1-3 lanes, limits {13,17,22}, signals 30 s + 3 s."""
    rng = np.random.default_rng(SEED_BASE + 2)
    N = grid * grid
    und = _grid_undirected(grid, grid)
    U = len(und)
    ulen = rng.integers(100, 401, U)
    ulanes = rng.choice([1, 2, 3], U, p=[0.5, 0.3, 0.2])
    ulim = np.array([0.0, 13.0, 17.0, 22.0])[ulanes]                # limit tied to lanes (fill-in)
    ef, et, length, lanes, vlim = _directed(und, ulen, ulanes, ulim)
    xy = np.stack([np.arange(N) % grid, np.arange(N) // grid], 1) * 250.0
    sig = _signal_arrays(rng, N, et, np.ones(N, bool), 60, 6)
    origins = rng.integers(0, N, n_vehicles)
    dests = (origins + rng.integers(1, N, n_vehicles)) % N
    depart = np.clip(rng.normal(1800.0, 600.0, n_vehicles), 0.0, None)
    v0m = rng.uniform(0.9, 1.1, n_vehicles)
    return _finish("cfg2_grid32", rng, N, ef, et, length, lanes, vlim, np.full(N, CTRL_SIGNAL),
                   sig, origins, dests, depart, steps, v0m, None, xy, workers)


def config3(n_vehicles=1_000_000, steps=43200, grid=256, n_origin_nodes=4096, workers=None,
            depart_mean_s=10800.0, depart_sd_s=3600.0, name="cfg3_perturbed256"):
    """configs[2]: perturbed grid, 5% of edges removed, arterial corridors, gravity OD,
    morning-peak departures (t=0 is 05:00, mean 08:00, sd 1 h).  Trips start at
    `n_origin_nodes` sampled nodes, mirroring the paper's zone-centroid -> nearest-node
    mapping; this also bounds the number of shortest-path trees."""
    rng = np.random.default_rng(SEED_BASE + 3)
    N0 = grid * grid
    spacing = 200.0
    gx, gy = np.arange(N0) % grid, np.arange(N0) // grid
    xy = np.stack([gx, gy], 1) * spacing + rng.uniform(-0.3, 0.3, (N0, 2)) * spacing
    und = _grid_undirected(grid, grid)
    period = max(2, min(32, grid // 2))
    on_art = lambda n: ((gx[n] % period) == period // 2, (gy[n] % period) == period // 2)
    ax0, ay0 = on_art(und[:, 0]); ax1, ay1 = on_art(und[:, 1])
    arterial = (ax0 & ax1 & (gx[und[:, 0]] == gx[und[:, 1]])) | (ay0 & ay1 & (gy[und[:, 0]] == gy[und[:, 1]]))
    removable = ~arterial
    drop = removable & (rng.random(len(und)) < 0.05)      # corridors stay whole
    und, arterial = und[~drop], arterial[~drop]
    U = len(und)
    ulanes = np.where(arterial, 4, rng.integers(1, 3, U))
    ulim = np.where(arterial, 29.0, 13.0)
    ulen = np.maximum(40, np.rint(np.hypot(*(xy[und[:, 0]] - xy[und[:, 1]]).T)).astype(np.int64))
    ef, et, length, lanes, vlim = _directed(und, ulen, ulanes, ulim)
    keep_node, remap, keep_edge = _largest_scc(N0, ef, et)
    ef, et = remap[ef[keep_edge]], remap[et[keep_edge]]
    length, lanes, vlim = length[keep_edge], lanes[keep_edge], vlim[keep_edge]
    xy = xy[keep_node]
    N = int(keep_node.sum())
    art_node = np.zeros(N, bool)
    art_node[ef[lanes == 4]] = True
    art_node[et[lanes == 4]] = True
    ctrl = np.where(art_node, CTRL_SIGNAL, CTRL_PRIORITY)
    sig = _signal_arrays(rng, N, et, art_node, 60, 6)
    n_on = min(n_origin_nodes, N)
    onodes = np.sort(rng.choice(N, n_on, replace=False))
    origins = np.sort(onodes[rng.integers(0, n_on, n_vehicles)])
    uo, cnt = np.unique(origins, return_counts=True)
    dests = _gravity_dests(rng, xy, uo, cnt, 5000.0)
    perm = rng.permutation(n_vehicles)                               # ids carry no spatial order
    origins, dests = origins[perm], dests[perm]
    horizon = steps * DEFAULT_PARAMS["dt"]
    depart = np.clip(rng.normal(depart_mean_s, depart_sd_s, n_vehicles), 0.0, horizon)
    v0m = rng.uniform(0.9, 1.1, n_vehicles)
    return _finish(name, rng, N, ef, et, length, lanes, vlim, ctrl, sig, origins, dests, depart,
                   steps, v0m, None, xy, workers)


def config4(n_vehicles=3_000_000, steps=172_800, n_points=1_000_000, side_m=100_000.0,
            n_centroids=4096, workers=None, name="cfg4_metro"):
    """configs[3] metro-scale synthetic: random planar road graph (Delaunay-derived) of ~1 M nodes /
    ~2.5 M directed edges with hierarchical classes, signals on nodes of degree >= 3, 3 M trips
    between `n_centroids` zone-centroid nodes with gravity OD and bimodal
    departures (t = 0 is midnight; Gaussians at 08:00 and 17:30, sd 1 h).  Everything scales with
    `n_points` / `side_m` for the small versions used in tests."""
    from scipy.spatial import Delaunay, cKDTree
    rng = np.random.default_rng(SEED_BASE + 4)
    pts = rng.random((int(n_points * 1.12), 2)) * side_m
    # minimum separation 30 m: drop the higher-numbered point of every too-close pair
    close = cKDTree(pts).query_pairs(30.0, output_type="ndarray")
    keep = np.ones(len(pts), bool)
    keep[close[:, 1]] = False
    pts = pts[keep][:n_points]
    N0 = len(pts)
    tri = Delaunay(pts).simplices
    # thin the Delaunay graph (~3 N edges) to ~1.25 N: drop the longest side of every triangle
    # (the Urquhart graph: planar, contains the Euclidean minimum spanning tree, so connected)
    sides = np.stack([tri[:, [0, 1]], tri[:, [1, 2]], tri[:, [2, 0]]], 1)            # [T, 3, 2]
    slen = np.hypot(*(pts[sides[..., 0]] - pts[sides[..., 1]]).transpose(2, 0, 1))   # [T, 3]
    longest = np.zeros(slen.shape, bool)
    longest[np.arange(len(tri)), np.argmax(slen, axis=1)] = True
    skey = np.minimum(sides[..., 0], sides[..., 1]).astype(np.int64) * N0 + np.maximum(sides[..., 0], sides[..., 1])
    drop = np.unique(skey[longest])
    allk = np.unique(skey)
    keepk = allk[~np.isin(allk, drop)]
    und = np.stack([keepk // N0, keepk % N0], 1)
    ulen = np.hypot(*(pts[und[:, 0]] - pts[und[:, 1]]).T)
    # hierarchy by distance of the edge midpoint to a coarse (freeway) and a fine (arterial) lattice
    mid = 0.5 * (pts[und[:, 0]] + pts[und[:, 1]])
    def lattice_dist(pitch):
        r = np.abs(((mid + 0.5 * pitch) % pitch) - 0.5 * pitch)
        return r.min(axis=1)
    d_fw, d_art = lattice_dist(side_m / 10.0), lattice_dist(side_m / 50.0)
    fw = d_fw <= np.quantile(d_fw, 0.02)
    art = ~fw & (d_art <= np.quantile(d_art[~fw], 0.15 / 0.98))
    ulanes = np.where(fw, 4, np.where(art, rng.integers(2, 4, len(und)), 1))
    ulim = np.where(fw, 29.0, np.where(art, 17.0, 11.0))
    ulen = np.maximum(40, np.rint(ulen)).astype(np.int64)
    ef, et, length, lanes, vlim = _directed(und, ulen, ulanes, ulim)
    keep_node, remap, keep_edge = _largest_scc(N0, ef, et)
    ef, et = remap[ef[keep_edge]], remap[et[keep_edge]]
    length, lanes, vlim = length[keep_edge], lanes[keep_edge], vlim[keep_edge]
    xy = pts[keep_node]
    N = int(keep_node.sum())
    n_in = np.bincount(et, minlength=N)
    sig_node = n_in >= 3
    ctrl = np.where(sig_node, CTRL_SIGNAL, CTRL_FREE)
    cycle = rng.integers(120, 241, N)                                  # 60..120 s at dt = 0.5 s
    green = np.maximum(1, cycle // np.maximum(1, n_in) - 6)            # all-red 6 steps per phase
    sig = _signal_arrays(rng, N, et, sig_node, green, 6)
    n_c = min(n_centroids, N)
    cent = np.sort(rng.choice(N, n_c, replace=False))
    o_idx = np.sort(rng.integers(0, n_c, n_vehicles))
    uo, cnt = np.unique(o_idx, return_counts=True)
    d_idx = _gravity_dests(rng, xy[cent], uo, cnt, 5000.0)             # gravity OD between centroids
    origins, dests = cent[o_idx], cent[d_idx]
    perm = rng.permutation(n_vehicles)
    origins, dests = origins[perm], dests[perm]
    horizon = steps * DEFAULT_PARAMS["dt"]
    am = rng.random(n_vehicles) < 0.5
    scale = horizon / 86400.0                                          # small versions compress the day
    depart = np.where(am, rng.normal(8.0 * 3600, 3600.0, n_vehicles), rng.normal(17.5 * 3600, 3600.0, n_vehicles))
    depart = np.clip(depart * scale, 0.0, horizon)
    v0m = rng.uniform(0.9, 1.1, n_vehicles)
    return _finish(name, rng, N, ef, et, length, lanes, vlim, ctrl, sig, origins, dests, depart,
                   steps, v0m, None, xy, workers)


def config5(n_vehicles=2_000_000, steps=28800, grid=256, core=8, workers=None):
    """configs[4] congestion stress: full grid, 2 lanes, 200 m, everyone leaves the central
    core x core nodes within 15 min for uniform destinations."""
    rng = np.random.default_rng(SEED_BASE + 5)
    N = grid * grid
    und = _grid_undirected(grid, grid)
    ef, et = _directed(und)
    E = len(ef)
    gx, gy = np.arange(N) % grid, np.arange(N) // grid
    xy = np.stack([gx, gy], 1) * 200.0
    lo = grid // 2 - core // 2
    central = np.nonzero((gx >= lo) & (gx < lo + core) & (gy >= lo) & (gy < lo + core))[0]
    origins = central[rng.integers(0, len(central), n_vehicles)]
    dests = (origins + rng.integers(1, N, n_vehicles)) % N
    depart = rng.random(n_vehicles) * 900.0
    z = np.zeros(N, np.uint32)
    return _finish("cfg5_stress", rng, N, ef, et, np.full(E, 200), np.full(E, 2), np.full(E, 15.0),
                   np.full(N, CTRL_PRIORITY), (z, z, z), origins, dests, depart, steps,
                   np.ones(n_vehicles), None, xy, workers)


def config3_dense(n_vehicles=1_000_000, steps=2400, workers=None):
    """DIAGNOSTIC, not a sixth config: config 3's network with every departure
    compressed into the first 60 s, so that ~1 M vehicles are active at once.  Separates kernel
    efficiency from the per-step latency floor."""
    return config3(n_vehicles=n_vehicles, steps=steps, workers=workers, depart_mean_s=30.0,
                   depart_sd_s=15.0, name="cfg3_dense_diagnostic")


def with_trucks(bundle, share=0.10, seed=0, name=None):
    """The same workload with a share of the vehicles turned into trucks."""
    rng = np.random.default_rng(SEED_BASE + 100 + seed)
    ty = (rng.random(bundle["n_vehicles"]) < share).astype(np.uint8)
    return dict(bundle, name=name or bundle["name"] + "_trucks", veh_type=ty,
                params=dict(bundle["params"], **TRUCK_PARAMS))


def with_controls(bundle, seed=0, amber_steps=6, name=None):
    """The same workload with the control variants of PAPER.md:402 mixed in: PRIORITY nodes become
    STOP nodes, half of the SIGNAL nodes get one phase per movement (n*m), every signal an amber."""
    rng = np.random.default_rng(SEED_BASE + 200 + seed)
    ctrl = np.array(bundle["node_ctrl"], np.uint8)
    ctrl[ctrl == CTRL_PRIORITY] = CTRL_STOP
    sig = np.nonzero(ctrl == CTRL_SIGNAL)[0]
    ctrl[sig[rng.random(len(sig)) < 0.5]] = CTRL_SIGNAL_NM
    return dict(bundle, name=name or bundle["name"] + "_controls", node_ctrl=ctrl,
                params=dict(bundle["params"], amber_steps=amber_steps, stop_dist=4.0, stop_speed=0.5))


# --------------------------------------------------------------------------- edge numbering

def spatial_edge_order(bundle, bits=16):
    """A space-filling (Morton / Z-curve) order of the edges by the midpoint of their end nodes:
    order[new id] = old id.  The simulator lays out edge records, atlas rows and claim words in the
    CALLER's edge order, so an edge numbering with spatial locality is what keeps a metro-scale network's
    gathers in L2 (config 4)."""
    xy = np.asarray(bundle["node_xy"], np.float64)
    mid = 0.5 * (xy[bundle["edge_from"]] + xy[bundle["edge_to"]])
    lo, hi = mid.min(0), mid.max(0)
    q = np.minimum(((mid - lo) / np.maximum(hi - lo, 1e-9) * (1 << bits)).astype(np.uint64), (1 << bits) - 1)
    code = np.zeros(len(mid), np.uint64)
    for k in range(bits):
        code |= ((q[:, 0] >> np.uint64(k)) & np.uint64(1)) << np.uint64(2 * k)
        code |= ((q[:, 1] >> np.uint64(k)) & np.uint64(1)) << np.uint64(2 * k + 1)
    return np.argsort(code, kind="stable").astype(np.uint32)


def renumber_edges(bundle, order, name=None):
    """The same network and demand with edge `order[n]` renamed `n` (edge arrays permuted, routes
    translated).  A different input as far as the simulators are concerned: ties that go by edge index
    (signal phase order, R16 / R35) fall differently, so its results are its own."""
    order = np.asarray(order, np.int64)
    new_id = np.empty(len(order), np.uint32)
    new_id[order] = np.arange(len(order), dtype=np.uint32)
    out = dict(bundle, name=name or bundle["name"] + "_renumbered")
    for k in ("edge_from", "edge_to", "edge_len_m", "edge_lanes", "edge_vlim"):
        out[k] = np.ascontiguousarray(bundle[k][order])
    out["route_edges"] = new_id[bundle["route_edges"]]
    return out


# --------------------------------------------------------------------------- re-routing inputs

REROUTE_SHARES = (1.0, 1.0, 0.5, 0.25)     # "all routes the first and second iteration, and
                                           # then we decay it to half and one-fourth of the vehicles"
W_UNIT = 256                               # routing weights are integers, 1/256 simulation step (R37)


def free_flow_weights(bundle):
    """The initial routing weights of PAPER.md:386, "estimating the travel time (t_t) of each edge as
    t_t = sqrt(edge_#lines) edge_length / edge_speed" -- read as length / (speed * sqrt(lanes)), the
    form under which "most vehicles ... use the highways" as that paragraph goes on to say (DESIGN.md
    reading R41) -- in the integer units the re-routing call takes.  An INPUT of ts_reroute."""
    b = bundle
    t = b["edge_len_m"].astype(np.float64) / (b["edge_vlim"].astype(np.float64) * np.sqrt(b["edge_lanes"].astype(np.float64)))
    return np.clip(np.rint(t / b["params"]["dt"] * W_UNIT), 1, 1 << 20).astype(np.uint32)


def reroute_mask(n_vehicles, iteration, seed=0):
    """Which vehicles recompute their path in iteration 0, 1, 2, 3: a seeded random
    subset of the stated share; an INPUT of ts_reroute."""
    share = REROUTE_SHARES[min(iteration, len(REROUTE_SHARES) - 1)]
    if share >= 1.0:
        return np.ones(n_vehicles, np.uint8)
    rng = np.random.default_rng(SEED_BASE + 300 + 17 * seed + iteration)
    return (rng.random(n_vehicles) < share).astype(np.uint8)


# --------------------------------------------------------------------------- static assignment inputs

def sue_inputs(bundle, horizon_s=3600.0):
    """Inputs of the static user equilibrium of PAPER.md:307-338 for a config's network and demand:
    free-flow time t0 = length / speed (Eq. 4), capacity per edge in vehicles per second
    from a per-lane hourly capacity by road class (Table 2 gives 800-2200 per lane per
    hour by OpenStreetMap type, which synthetic edges do not have: 2200 for >= 4 lanes, 1000 for a
    limit >= 17 m/s, else 900), and the OD matrix as integer trips per (origin node, destination
    node) pair, the demand rate being trips per `horizon_s`."""
    b = bundle
    t0 = b["edge_len_m"].astype(np.float64) / b["edge_vlim"].astype(np.float64)
    per_lane = np.where(b["edge_lanes"] >= 4, 2200.0, np.where(b["edge_vlim"] >= 17.0, 1000.0, 900.0))
    cap = per_lane * b["edge_lanes"].astype(np.float64) / 3600.0
    off = b["route_off"].astype(np.int64)
    o = b["edge_from"][b["route_edges"][off[:-1]]].astype(np.int64)
    d = b["edge_to"][b["route_edges"][off[1:] - 1]].astype(np.int64)
    key, trips = np.unique(o * b["n_nodes"] + d, return_counts=True)
    return dict(t0=t0, cap=cap * horizon_s, od_origin=(key // b["n_nodes"]).astype(np.uint32),
                od_dest=(key % b["n_nodes"]).astype(np.uint32), od_trips=trips.astype(np.uint32))


_BY_NAME = {
    "cfg1": config1, "cfg2": config2, "cfg3": config3, "cfg4": config4, "cfg5": config5,
    "cfg3_dense": config3_dense,
    # config 4's network and demand with its edges numbered along a space-filling curve (diagnostic: DESIGN.md section 6)
    "cfg4_morton": lambda: (lambda b: renumber_edges(b, spatial_edge_order(b), "cfg4_metro_morton"))(config4()),
    "cfg4_small_morton": lambda: (lambda b: renumber_edges(b, spatial_edge_order(b), "cfg4_small_morton"))(
        config4(n_vehicles=60_000, steps=7200, n_points=20_000, side_m=14_000.0, n_centroids=256, name="cfg4_small")),
    # SURVEY.md 8(f) rows 3 and 4 on config 2's network and demand
    "cfg2_trucks": lambda: with_trucks(config2()),
    "cfg2_controls": lambda: with_controls(config2()),
    "cfg2_trucks_controls": lambda: with_controls(with_trucks(config2())),
    # quick functional checks, not reported workloads
    "cfg3_small": lambda: config3(n_vehicles=50_000, steps=7200, grid=64, n_origin_nodes=512,
                                  depart_mean_s=1200.0, depart_sd_s=400.0, name="cfg3_small"),
    "cfg4_small": lambda: config4(n_vehicles=60_000, steps=7200, n_points=20_000, side_m=14_000.0,
                                  n_centroids=256, name="cfg4_small"),
    "cfg5_small": lambda: config5(n_vehicles=60_000, steps=7200, grid=48, core=4),
}


def by_name(name):
    """Workload bundle by short name (bench.py --workload, tests/golden/make_golden.py)."""
    if name not in _BY_NAME:
        raise KeyError(f"unknown workload {name!r}; known: {sorted(_BY_NAME)}")
    return _BY_NAME[name]()
