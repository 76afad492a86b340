"""ORACLE -- test infrastructure, not product code.

ctypes wrapper around oracle/ts_oracle.c (the plain single-threaded CPU restatement of the
paper's per-vehicle traffic microsimulation).  Only tests/,
__graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may import this
package; nothing under paper_1807_01148_b200/ does, and this package imports nothing from it.
"""
from __future__ import annotations

import ctypes as C

import numpy as np

from .build import build as _build

_PARAM_FIELDS = [
    ("dt", C.c_float), ("a", C.c_float), ("b", C.c_float), ("T", C.c_float), ("s0", C.c_float),
    ("veh_len", C.c_float), ("b_safe", C.c_float), ("politeness", C.c_float),
    ("lc_threshold", C.c_float), ("mand_dist_default", C.c_float),
    ("lookahead_cells", C.c_uint32), ("lookback_cells", C.c_uint32), ("lc_period", C.c_uint32),
    ("entry_zone_cells", C.c_uint32), ("insert_clear_cells", C.c_uint32),
    ("sample_period_steps", C.c_uint32), ("emissions", C.c_uint32),
    ("n_types", C.c_uint32), ("type_len", C.c_float * 4), ("type_a", C.c_float * 4),
    ("type_vmax", C.c_float * 4), ("amber_steps", C.c_uint32), ("stop_dist", C.c_float),
    ("stop_speed", C.c_float),
]
# fields that may be absent from a params dict, with the value that switches the feature off
_OPTIONAL = dict(emissions=0, n_types=0, type_len=(), type_a=(), type_vmax=(), amber_steps=0,
                 stop_dist=4.0, stop_speed=0.5)


class OrcParams(C.Structure):
    _fields_ = _PARAM_FIELDS


_COUNTER_NAMES = ["updates", "own_cells", "next_cells", "lc_evals", "lc_cells", "lc_accepts",
                  "lc_mandatory", "crossings", "cross_lost", "held_red", "cap_bound",
                  "departures", "arrivals", "peak_active", "own_chunks16", "next_chunks16", "lc_chunks16"]


class OrcCounters(C.Structure):
    _fields_ = [(n, C.c_uint64) for n in _COUNTER_NAMES]


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_build())
        L.orc_create.restype = C.c_void_p
        L.orc_create.argtypes = [C.c_uint32, C.c_uint32] + [C.c_void_p] * 9 + [C.c_uint32] + [C.c_void_p] * 6 + [C.POINTER(OrcParams)]
        L.orc_step.restype = C.c_int
        L.orc_step.argtypes = [C.c_void_p, C.c_uint32, C.c_void_p, C.c_int, C.c_uint64]
        L.orc_read_state.restype = None
        L.orc_read_state.argtypes = [C.c_void_p] * 14
        L.orc_read_edge_stats.restype = None
        L.orc_read_edge_stats.argtypes = [C.c_void_p] * 7 + [C.c_int]
        L.orc_read_emissions.restype = None
        L.orc_read_emissions.argtypes = [C.c_void_p] * 3
        L.orc_co_rate.restype = C.c_float
        L.orc_co_rate.argtypes = [C.c_float]
        L.orc_fuel_rate.restype = C.c_float
        L.orc_fuel_rate.argtypes = [C.c_float, C.c_float]
        L.orc_get_counters.restype = None
        L.orc_get_counters.argtypes = [C.c_void_p, C.POINTER(OrcCounters)]
        L.orc_set_threads.restype = None
        L.orc_set_threads.argtypes = [C.c_void_p, C.c_int]
        L.orc_destroy.restype = None
        L.orc_destroy.argtypes = [C.c_void_p]
        L.orc_last_error.restype = C.c_char_p
        L.orc_idm.restype = C.c_float
        L.orc_idm.argtypes = [C.POINTER(OrcParams), C.c_float, C.c_float, C.c_int, C.c_float, C.c_float]
        L.orc_speed_code.restype = C.c_uint8
        L.orc_speed_code.argtypes = [C.c_float]
        L.orc_speed_decode.restype = C.c_float
        L.orc_speed_decode.argtypes = [C.c_uint8]
        L.orc_signal_green.restype = C.c_int
        L.orc_signal_green.argtypes = [C.c_uint32] * 5 + [C.c_uint64]
        L.orc_signal_phase.restype = C.c_int
        L.orc_signal_phase.argtypes = [C.c_uint32] * 8 + [C.c_uint64]
        L.orc_mix64.restype = C.c_uint64
        L.orc_mix64.argtypes = [C.c_uint64]
        _lib = L
    return _lib


def make_params(d) -> OrcParams:
    p = OrcParams()
    for name, ctype in _PARAM_FIELDS:
        val = d.get(name, _OPTIONAL[name]) if name in _OPTIONAL else d[name]
        if name.startswith("type_"):
            val = ctype(*[float(x) for x in val])
        setattr(p, name, val)
    return p


def _ptr(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


class OracleError(RuntimeError):
    pass


class Oracle:
    """One simulation.  `bundle` is a dict as produced by the workload module."""

    def __init__(self, bundle):
        L = lib()
        b = bundle
        self.V, self.E = int(b["n_vehicles"]), int(b["n_edges"])
        self._p = make_params(b["params"])
        self._keep = [np.ascontiguousarray(b[k]) for k in (
            "edge_from", "edge_to", "edge_len_m", "edge_lanes", "edge_vlim", "node_ctrl",
            "sig_green_steps", "sig_allred_steps", "sig_offset_steps", "route_off", "route_edges",
            "depart_time_s", "v0_mult", "mand_dist_m")]
        self._keep.append(None if b.get("veh_type") is None else np.ascontiguousarray(b["veh_type"], np.uint8))
        k = self._keep
        self._h = L.orc_create(int(b["n_nodes"]), self.E, *[_ptr(a) for a in k[:9]], self.V,
                               *[_ptr(a) for a in k[9:]], C.byref(self._p))
        if not self._h:
            raise OracleError(L.orc_last_error().decode())

    def set_threads(self, n):
        """Host threads for the intent loop (results do not depend on it; default 1)."""
        lib().orc_set_threads(self._h, int(n))

    def step(self, n, digests=False, check=0, order_seed=0):
        d = np.zeros(n, np.uint64) if digests else None
        if lib().orc_step(self._h, int(n), _ptr(d), int(check), int(order_seed)) != 0:
            raise OracleError(lib().orc_last_error().decode())
        return d

    def read_state(self):
        V = self.V
        out = dict(status=np.zeros(V, np.uint8), edge=np.zeros(V, np.uint32), lane=np.zeros(V, np.uint8),
                   cell=np.zeros(V, np.uint32), x=np.zeros(V, np.float32), v=np.zeros(V, np.float32),
                   route_idx=np.zeros(V, np.uint32), insert_step=np.zeros(V, np.uint32),
                   arrive_step=np.zeros(V, np.uint32))
        step = C.c_uint64(); npend = C.c_uint32(); nact = C.c_uint32(); narr = C.c_uint32()
        lib().orc_read_state(self._h, *[_ptr(out[k]) for k in ("status", "edge", "lane", "cell", "x", "v", "route_idx", "insert_step", "arrive_step")],
                             C.addressof(step), C.addressof(npend), C.addressof(nact), C.addressof(narr))
        out.update(step=step.value, n_pending=npend.value, n_active=nact.value, n_arrived=narr.value)
        return out

    def read_counts(self):
        """Scalars only."""
        step = C.c_uint64(); npend = C.c_uint32(); nact = C.c_uint32(); narr = C.c_uint32()
        lib().orc_read_state(self._h, *([None] * 9), C.addressof(step), C.addressof(npend),
                             C.addressof(nact), C.addressof(narr))
        return dict(step=step.value, n_pending=npend.value, n_active=nact.value, n_arrived=narr.value)

    def read_edge_stats(self, reset=False):
        E = self.E
        out = dict(entered=np.zeros(E, np.uint32), exited=np.zeros(E, np.uint32),
                   exit_steps_sum=np.zeros(E, np.uint64), sample_count_sum=np.zeros(E, np.uint32),
                   sample_speedcode_sum=np.zeros(E, np.uint64))
        ns = C.c_uint32()
        lib().orc_read_edge_stats(self._h, *[_ptr(out[k]) for k in ("entered", "exited", "exit_steps_sum", "sample_count_sum", "sample_speedcode_sum")],
                                  C.addressof(ns), int(bool(reset)))
        out["n_samples"] = ns.value
        return out

    def read_emissions(self):
        """Per-vehicle grams of CO (Eq. 8) and millilitres of fuel (Eq. 9) since step 0."""
        out = dict(co_g=np.zeros(self.V, np.float32), fuel_ml=np.zeros(self.V, np.float32))
        lib().orc_read_emissions(self._h, _ptr(out["co_g"]), _ptr(out["fuel_ml"]))
        return out

    def counters(self):
        c = OrcCounters()
        lib().orc_get_counters(self._h, C.byref(c))
        return {n: getattr(c, n) for n in _COUNTER_NAMES}

    def close(self):
        if self._h:
            lib().orc_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def co_rate(v):
    return float(lib().orc_co_rate(v))


def fuel_rate(v, acc):
    return float(lib().orc_fuel_rate(v, acc))


def idm(params, v, v0, has_leader, s, dv):
    return float(lib().orc_idm(C.byref(make_params(params)), v, v0, int(has_leader), s, dv))


def utilisation(edge_stats, bundle):
    """"the number of vehicles at the sampling time divided by the maximum number of
    vehicles that can fit on the edge ... the length of the edge times the number of lines divided by
    the average length of a vehicle plus the lead gap" (vehicle length of type 0, lead gap s0), averaged
    over the samples taken; and the mean sampled speed in m/s.  fp64."""
    p = bundle["params"]
    cap = bundle["edge_len_m"].astype(np.float64) * bundle["edge_lanes"] / (p["veh_len"] + p["s0"])
    n = int(edge_stats["n_samples"])
    cnt = edge_stats["sample_count_sum"].astype(np.float64)
    util = cnt / n / cap if n else np.zeros_like(cap)
    speed = np.where(cnt > 0, edge_stats["sample_speedcode_sum"] * 0.25 / np.maximum(cnt, 1), 0.0)
    return util, speed
