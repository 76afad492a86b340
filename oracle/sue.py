"""ORACLE -- test infrastructure, not product code.

Static user equilibrium by the Frank-Wolfe algorithm with BPR travel times, PAPER.md:307-338
(section 5.3, Eq. 6) and PAPER.md:200-216 (Eq. 3: t = t0 (1 + alpha (v/c)^beta), alpha = 0.15,
beta = 4).  Plain numpy in fp64, step by step in the paper's order:

  1. x_0 = all-or-nothing assignment on the free-flow times                  (PAPER.md:331 step 1)
  2. y_k = argmin over feasible flows of grad f(x_k) . y = all-or-nothing assignment on t(x_k)
                                                                              (step 2)
  3. step length a_k in [0, 1] with f((1 - a) x_k + a y_k) <= f(x_k): the minimiser along the
     segment, found by bisection on the derivative g(a) = sum_e (y_e - x_e) t_e(x_e + a (y_e - x_e))
                                                                              (step 3)
  4. x_{k+1} = (1 - a_k) x_k + a_k y_k                                        (step 4)

with f(x) = sum_e integral_0^{x_e} t_e(s) ds = sum_e t0_e (x_e + alpha x_e^5 / (5 c_e^4))  (Eq. 6).

Readings (R42-R44): beta is the integer 4 (two squarings); the all-or-nothing step uses
shortest paths on INTEGER weights w_e = rint(t_e * weight_scale) clamped to [1, 2^20] with the tie-break of the
re-routing oracle (oracle/reroute.py, R38), so that the discrete part of the iteration does not hang
on floating-point ties; demand is integer trips per OD pair.
Only tests/ and bench.py's oracle legs may import this module; it imports nothing from the package.
"""
from __future__ import annotations

import numpy as np

from .reroute import shortest_path_trees

ALPHA, BETA = 0.15, 4


def bpr_time(t0, cap, x, alpha=ALPHA):
    """Eq. 3 with beta = 4."""
    r = x / cap
    r2 = r * r
    return t0 * (1.0 + alpha * (r2 * r2))


def objective(t0, cap, x, alpha=ALPHA):
    """Eq. 6: sum of the integrals of the BPR curves."""
    r = x / cap
    r2 = r * r
    return float(np.sum(t0 * (x + (alpha / 5.0) * (x * (r2 * r2)))))


def weights(t, weight_scale):
    return np.clip(np.rint(t * weight_scale), 1, 1 << 20).astype(np.uint32)


def all_or_nothing(n_nodes, edge_from, edge_to, w, od_origin, od_dest, od_trips):
    """Every OD pair's trips on its shortest path (tie-break R38).  Integer flows per edge."""
    ef = np.asarray(edge_from, np.int64)
    y = np.zeros(len(ef), np.uint64)
    origins = np.unique(od_origin)
    for lo in range(0, len(origins), 64):
        src = origins[lo:lo + 64]
        dist, pred = shortest_path_trees(n_nodes, edge_from, edge_to, w, src)
        row_of = {int(s): r for r, s in enumerate(src)}
        for q in np.nonzero(np.isin(od_origin, src))[0]:
            o, d, trips = int(od_origin[q]), int(od_dest[q]), int(od_trips[q])
            r = row_of[o]
            if o == d or not np.isfinite(dist[r, d]):
                continue
            v = d
            while v != o:
                e = int(pred[r, v])
                y[e] += np.uint64(trips)
                v = int(ef[e])
    return y


def solve(n_nodes, edge_from, edge_to, t0, cap, od_origin, od_dest, od_trips, iterations=20,
          bisections=40, weight_scale=1000.0, alpha=ALPHA):
    t0 = np.asarray(t0, np.float64); cap = np.asarray(cap, np.float64)
    aon = lambda t: all_or_nothing(n_nodes, edge_from, edge_to, weights(t, weight_scale), od_origin, od_dest,
                                   od_trips).astype(np.float64)
    x = aon(t0)
    hist = dict(objective=[objective(t0, cap, x, alpha)], step=[], gap=[])
    for _ in range(iterations):
        t = bpr_time(t0, cap, x, alpha)
        y = aon(t)
        d = y - x
        hist["gap"].append(float((np.sum(x * t) - np.sum(y * t)) / np.sum(x * t)))
        g = lambda a: float(np.sum(d * bpr_time(t0, cap, x + a * d, alpha)))
        if g(1.0) <= 0.0:
            a = 1.0
        elif g(0.0) >= 0.0:
            a = 0.0
        else:
            lo, hi = 0.0, 1.0
            for _ in range(bisections):
                mid = 0.5 * (lo + hi)
                if g(mid) > 0.0:
                    hi = mid
                else:
                    lo = mid
            a = 0.5 * (lo + hi)
        x = x + a * d
        hist["step"].append(a)
        hist["objective"].append(objective(t0, cap, x, alpha))
    return x, bpr_time(t0, cap, x, alpha), hist
