"""Thin ctypes binding of libts.so (include/trafficsim.h): argument marshalling only.

PyTorch is used for what the header asks the caller to provide: one device workspace tensor
and a CUDA stream.  Every step of the simulation runs in the library's kernels; there is no
Python or CPU fallback, and loading fails loudly if the library has not been built."""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libts.so")

TS_OK, TS_EINVAL, TS_ENOMEM, TS_ECUDA, TS_EINVARIANT = 0, -1, -2, -3, -4

EXPORTS = ["ts_query_workspace", "ts_create", "ts_step", "ts_step_digest", "ts_reset",
           "ts_read_state", "ts_read_edge_stats", "ts_set_option", "ts_read_profile",
           "ts_read_emissions", "ts_read_utilisation", "ts_reroute", "ts_read_routes", "ts_sue_workspace", "ts_sue_solve", "ts_sssp_static", "ts_sssp_static_max_nodes", "ts_checkpoint_size", "ts_checkpoint", "ts_restore", "ts_destroy", "ts_last_error", "ts_version"]

_u32p, _u8p, _f32p, _u64p = (C.POINTER(C.c_uint32), C.POINTER(C.c_uint8), C.POINTER(C.c_float),
                             C.POINTER(C.c_uint64))


class TsNetwork(C.Structure):
    _fields_ = [("n_nodes", C.c_uint32), ("n_edges", C.c_uint32), ("edge_from", C.c_void_p),
                ("edge_to", C.c_void_p), ("edge_len_m", C.c_void_p), ("edge_lanes", C.c_void_p),
                ("edge_vlim", C.c_void_p), ("node_ctrl", C.c_void_p), ("sig_green_steps", C.c_void_p),
                ("sig_allred_steps", C.c_void_p), ("sig_offset_steps", C.c_void_p)]


class TsRoutes(C.Structure):
    _fields_ = [("n_vehicles", C.c_uint32), ("route_off", C.c_void_p), ("route_edges", C.c_void_p)]


class TsDepartures(C.Structure):
    _fields_ = [("depart_time_s", C.c_void_p), ("v0_mult", C.c_void_p), ("mand_dist_m", C.c_void_p),
                ("veh_type", C.c_void_p)]


class TsParams(C.Structure):
    _fields_ = [(n, C.c_float) for n in ("dt", "a", "b", "T", "s0", "veh_len", "b_safe", "politeness",
                                         "lc_threshold", "mand_dist_default")] + \
               [(n, C.c_uint32) for n in ("lookahead_cells", "lookback_cells", "lc_period",
                                          "entry_zone_cells", "insert_clear_cells", "sample_period_steps",
                                          "emissions", "n_types")] + \
               [("type_len", C.c_float * 4), ("type_a", C.c_float * 4), ("type_vmax", C.c_float * 4),
                ("amber_steps", C.c_uint32), ("stop_dist", C.c_float), ("stop_speed", C.c_float),
                ("route_capacity", C.c_uint32)]


# ts_params fields a bundle may leave out, with the value that switches the feature off
_OPTIONAL = dict(emissions=0, n_types=0, type_len=(), type_a=(), type_vmax=(), amber_steps=0,
                 stop_dist=4.0, stop_speed=0.5, route_capacity=0)


class TsDevice(C.Structure):
    _fields_ = [("workspace", C.c_void_p), ("bytes", C.c_size_t), ("cuda_stream", C.c_void_p),
                ("out_on_device", C.c_int)]


class TsStateOut(C.Structure):
    _fields_ = [(n, C.c_void_p) for n in ("status", "edge", "lane", "cell", "x", "v", "route_idx",
                                          "insert_step", "arrive_step")] + \
               [("step", C.c_uint64), ("n_pending", C.c_uint32), ("n_active", C.c_uint32),
                ("n_arrived", C.c_uint32), ("vehicle_updates", C.c_uint64)]


class TsEdgeStatsOut(C.Structure):
    _fields_ = [(n, C.c_void_p) for n in ("entered", "exited", "exit_steps_sum", "sample_count_sum",
                                          "sample_speedcode_sum")] + [("n_samples", C.c_uint32)]


class TsRerouteOut(C.Structure):
    _fields_ = [("n_rerouted", C.c_uint32), ("n_trees", C.c_uint32), ("route_entries", C.c_uint64),
                ("sssp_ms", C.c_float), ("device_ms", C.c_float), ("w", C.c_void_p)]


class TsSueProblem(C.Structure):
    _fields_ = [("n_nodes", C.c_uint32), ("n_edges", C.c_uint32), ("edge_from", C.c_void_p), ("edge_to", C.c_void_p),
                ("t0", C.c_void_p), ("cap", C.c_void_p), ("n_od", C.c_uint32), ("od_origin", C.c_void_p),
                ("od_dest", C.c_void_p), ("od_trips", C.c_void_p), ("alpha", C.c_double), ("weight_scale", C.c_double),
                ("iterations", C.c_uint32), ("bisections", C.c_uint32)]


class TsSueOut(C.Structure):
    _fields_ = [(n, C.c_void_p) for n in ("flow", "time", "objective", "gap", "step")] + \
               [("device_ms", C.c_float), ("sssp_ms", C.c_float), ("n_trees", C.c_uint32)]


class TsError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"ts error {code}: {msg}")
        self.code = code


_lib = None


def load():
    """dlopen libts.so.  No fallback: a missing library is an error."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} is not built: run `python -m paper_1807_01148_b200.build` "
                              "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        L.ts_query_workspace.argtypes = [C.c_void_p] * 4 + [C.POINTER(C.c_size_t)]
        L.ts_create.argtypes = [C.c_void_p] * 5 + [C.POINTER(C.c_void_p)]
        L.ts_step.argtypes = [C.c_void_p, C.c_uint32]
        L.ts_step_digest.argtypes = [C.c_void_p, C.c_uint32, C.c_void_p]
        L.ts_reset.argtypes = [C.c_void_p]
        L.ts_read_state.argtypes = [C.c_void_p, C.c_void_p]
        L.ts_read_edge_stats.argtypes = [C.c_void_p, C.c_void_p, C.c_int]
        L.ts_set_option.argtypes = [C.c_void_p, C.c_char_p, C.c_longlong]
        L.ts_read_profile.argtypes = [C.c_void_p, C.c_void_p]
        L.ts_read_emissions.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.ts_reroute.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.ts_read_routes.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.POINTER(C.c_uint64)]
        L.ts_destroy.argtypes = [C.c_void_p]
        L.ts_destroy.restype = None
        L.ts_last_error.restype = C.c_char_p
        L.ts_version.restype = C.c_char_p
        L.ts_checkpoint_size.argtypes = [C.c_void_p, C.POINTER(C.c_size_t)]
        L.ts_checkpoint.argtypes = [C.c_void_p, C.c_void_p]
        L.ts_restore.argtypes = [C.c_void_p, C.c_void_p]
        for n in ("ts_checkpoint_size", "ts_checkpoint", "ts_restore"):
            getattr(L, n).restype = C.c_int
        L.ts_sssp_static.argtypes = [C.c_uint32, C.c_uint32] + [C.c_void_p] * 5 + [C.c_uint32] + [C.c_void_p] * 3
        L.ts_sssp_static.restype = C.c_int
        L.ts_sssp_static_max_nodes.restype = C.c_uint32
        L.ts_sue_workspace.argtypes = [C.c_void_p, C.POINTER(C.c_size_t)]
        L.ts_sue_solve.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.ts_read_utilisation.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        for n in EXPORTS[:15]:
            getattr(L, n).restype = C.c_int
        _lib = L
    return _lib


def _check(rc):
    if rc != 0:
        raise TsError(rc, load().ts_last_error().decode())


def _p(a):
    return None if a is None else a.ctypes.data


def marshal(bundle):
    """bundle dict -> (net, routes, dep, params, keepalive)."""
    b = bundle
    keep = {k: np.ascontiguousarray(b[k]) for k in (
        "edge_from", "edge_to", "edge_len_m", "edge_lanes", "edge_vlim", "node_ctrl",
        "sig_green_steps", "sig_allred_steps", "sig_offset_steps", "route_off", "route_edges",
        "depart_time_s")}
    for k in ("v0_mult", "mand_dist_m"):
        keep[k] = None if b.get(k) is None else np.ascontiguousarray(b[k])
    keep["veh_type"] = None if b.get("veh_type") is None else np.ascontiguousarray(b["veh_type"], np.uint8)
    net = TsNetwork(int(b["n_nodes"]), int(b["n_edges"]), *[_p(keep[k]) for k in (
        "edge_from", "edge_to", "edge_len_m", "edge_lanes", "edge_vlim", "node_ctrl",
        "sig_green_steps", "sig_allred_steps", "sig_offset_steps")])
    routes = TsRoutes(int(b["n_vehicles"]), _p(keep["route_off"]), _p(keep["route_edges"]))
    dep = TsDepartures(_p(keep["depart_time_s"]), _p(keep["v0_mult"]), _p(keep["mand_dist_m"]),
                       _p(keep["veh_type"]))
    vals = {}
    for n, ctype in TsParams._fields_:
        v = b["params"].get(n, _OPTIONAL[n]) if n in _OPTIONAL else b["params"][n]
        vals[n] = ctype(*[float(x) for x in v]) if n.startswith("type_") else v
    prm = TsParams(**vals)
    return net, routes, dep, prm, keep


def query_workspace(bundle) -> int:
    net, routes, dep, prm, _keep = marshal(bundle)
    n = C.c_size_t()
    _check(load().ts_query_workspace(C.byref(net), C.byref(routes), C.byref(dep), C.byref(prm), C.byref(n)))
    return n.value


class Sim:
    """ts_create / ts_step / ts_read_state / ts_read_edge_stats on one GPU."""

    def __init__(self, bundle, device="cuda:0", stream=None, mode=None):
        import torch
        L = load()
        self.V, self.E = int(bundle["n_vehicles"]), int(bundle["n_edges"])
        net, routes, dep, prm, keep = marshal(bundle)
        self.workspace_bytes = query_workspace(bundle)
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        self._ws = torch.empty(self.workspace_bytes + 256, dtype=torch.uint8, device=self.device)
        base = (self._ws.data_ptr() + 255) & ~255
        self._stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        dev = TsDevice(base, self.workspace_bytes, self._stream.cuda_stream, 0)
        h = C.c_void_p()
        _check(L.ts_create(C.byref(net), C.byref(routes), C.byref(dep), C.byref(prm), C.byref(dev), C.byref(h)))
        self._h = h
        if mode is not None:
            self.set_option("mode", mode)

    def set_option(self, key, value):
        _check(load().ts_set_option(self._h, key.encode(), int(value)))

    def step(self, n):
        _check(load().ts_step(self._h, int(n)))

    def step_digest(self, n):
        d = np.zeros(int(n), np.uint64)
        _check(load().ts_step_digest(self._h, int(n), d.ctypes.data))
        return d

    def reset(self):
        _check(load().ts_reset(self._h))

    def read_state(self):
        V = self.V
        out = dict(status=np.zeros(V, np.uint8), edge=np.zeros(V, np.uint32), lane=np.zeros(V, np.uint8),
                   cell=np.zeros(V, np.uint32), x=np.zeros(V, np.float32), v=np.zeros(V, np.float32),
                   route_idx=np.zeros(V, np.uint32), insert_step=np.zeros(V, np.uint32),
                   arrive_step=np.zeros(V, np.uint32))
        o = TsStateOut(*[_p(out[k]) for k in ("status", "edge", "lane", "cell", "x", "v", "route_idx",
                                               "insert_step", "arrive_step")])
        _check(load().ts_read_state(self._h, C.byref(o)))
        out.update(step=o.step, n_pending=o.n_pending, n_active=o.n_active, n_arrived=o.n_arrived,
                   vehicle_updates=o.vehicle_updates)
        return out

    def read_utilisation(self):
        """ts_read_utilisation: per-edge utilisation and mean sampled speed."""
        u, v = np.zeros(self.E, np.float32), np.zeros(self.E, np.float32)
        _check(load().ts_read_utilisation(self._h, u.ctypes.data, v.ctypes.data))
        return u, v

    def reroute(self, w_free, mask=None):
        """ts_reroute: new routes for the masked vehicles from the edge statistics accumulated so far
        (PAPER.md:386); resets the simulation.  Returns counts, device times and the weights used."""
        w_free = np.ascontiguousarray(w_free, np.uint32)
        m = None if mask is None else np.ascontiguousarray(mask, np.uint8)
        w = np.zeros(self.E, np.uint32)
        o = TsRerouteOut(w=w.ctypes.data)
        _check(load().ts_reroute(self._h, w_free.ctypes.data, None if m is None else m.ctypes.data, C.byref(o)))
        return dict(n_rerouted=o.n_rerouted, n_trees=o.n_trees, route_entries=o.route_entries,
                    sssp_ms=o.sssp_ms, device_ms=o.device_ms, w=w)

    def read_routes(self):
        """ts_read_routes: (route_off [V+1] uint64, route_edges uint32) of the routes in use."""
        n = C.c_uint64()
        _check(load().ts_read_routes(self._h, None, None, C.byref(n)))
        off = np.zeros(self.V + 1, np.uint64)
        edges = np.zeros(int(n.value), np.uint32)
        _check(load().ts_read_routes(self._h, off.ctypes.data, edges.ctypes.data, C.byref(n)))
        return off, edges

    def checkpoint(self):
        """ts_checkpoint: the whole state as one host byte array (numpy uint8)."""
        n = C.c_size_t()
        _check(load().ts_checkpoint_size(self._h, C.byref(n)))
        buf = np.empty(n.value, np.uint8)
        _check(load().ts_checkpoint(self._h, buf.ctypes.data))
        return buf

    def restore(self, buf):
        """ts_restore: back to the state of a checkpoint of a simulation created from the same inputs."""
        buf = np.ascontiguousarray(buf, np.uint8)
        _check(load().ts_restore(self._h, buf.ctypes.data))

    def read_counts(self):
        """Scalars only (no per-vehicle arrays are copied)."""
        o = TsStateOut()
        _check(load().ts_read_state(self._h, C.byref(o)))
        return dict(step=o.step, n_pending=o.n_pending, n_active=o.n_active, n_arrived=o.n_arrived,
                    vehicle_updates=o.vehicle_updates)

    def read_profile(self):
        """Option "profile": nanoseconds per simulation step in each phase, mean over the CTAs."""
        a = np.zeros(8, np.uint64)
        _check(load().ts_read_profile(self._h, a.ctypes.data))
        n = max(1, int(a[6]))
        names = ("phase1", "barrier1", "phase2", "barrier2", "sort", "digest")
        out = {k: float(a[i]) / n for i, k in enumerate(names)}
        out["phase1_slowest_cta"] = float(a[7]) / n     # per launch; meaningful after one ts_step call
        out["steps"] = int(a[6])
        return out

    def read_edge_stats(self, reset=False):
        E = self.E
        out = dict(entered=np.zeros(E, np.uint32), exited=np.zeros(E, np.uint32),
                   exit_steps_sum=np.zeros(E, np.uint64), sample_count_sum=np.zeros(E, np.uint32),
                   sample_speedcode_sum=np.zeros(E, np.uint64))
        o = TsEdgeStatsOut(*[_p(out[k]) for k in ("entered", "exited", "exit_steps_sum",
                                                   "sample_count_sum", "sample_speedcode_sum")])
        _check(load().ts_read_edge_stats(self._h, C.byref(o), int(bool(reset))))
        out["n_samples"] = o.n_samples
        return out

    def read_emissions(self):
        """Per-vehicle grams of CO (Eq. 8) and millilitres of fuel (Eq. 9)
        since step 0; the simulation must have been created with params["emissions"] != 0."""
        out = dict(co_g=np.zeros(self.V, np.float32), fuel_ml=np.zeros(self.V, np.float32))
        _check(load().ts_read_emissions(self._h, _p(out["co_g"]), _p(out["fuel_ml"])))
        return out

    def close(self):
        if getattr(self, "_h", None):
            load().ts_destroy(self._h)
            self._h = None
            self._ws = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def sue_solve(n_nodes, edge_from, edge_to, t0, cap, od_origin, od_dest, od_trips, iterations=20, bisections=40,
              weight_scale=1000.0, alpha=0.15, device="cuda:0"):
    """ts_sue_solve: static user equilibrium by Frank-Wolfe with BPR times.
    Marshalling only; returns (flow, time, dict(objective, gap, step, device_ms, sssp_ms, n_trees))."""
    import torch
    L = load()
    u32 = lambda a: np.ascontiguousarray(a, np.uint32)
    f64 = lambda a: np.ascontiguousarray(a, np.float64)
    keep = [u32(edge_from), u32(edge_to), f64(t0), f64(cap), u32(od_origin), u32(od_dest), u32(od_trips)]
    E, n_od = len(keep[0]), len(keep[4])
    prob = TsSueProblem(int(n_nodes), E, keep[0].ctypes.data, keep[1].ctypes.data, keep[2].ctypes.data,
                        keep[3].ctypes.data, n_od, keep[4].ctypes.data, keep[5].ctypes.data, keep[6].ctypes.data,
                        float(alpha), float(weight_scale), int(iterations), int(bisections))
    n = C.c_size_t()
    _check(L.ts_sue_workspace(C.byref(prob), C.byref(n)))
    dev_t = torch.device(device)
    torch.cuda.set_device(dev_t)
    ws = torch.empty(n.value + 256, dtype=torch.uint8, device=dev_t)
    base = (ws.data_ptr() + 255) & ~255
    dev = TsDevice(base, n.value, torch.cuda.current_stream(dev_t).cuda_stream, 0)
    flow, time_ = np.zeros(E), np.zeros(E)
    obj, gap, step = np.zeros(iterations + 1), np.zeros(iterations), np.zeros(iterations)
    out = TsSueOut(flow.ctypes.data, time_.ctypes.data, obj.ctypes.data, gap.ctypes.data, step.ctypes.data)
    _check(L.ts_sue_solve(C.byref(prob), C.byref(dev), C.byref(out)))
    return flow, time_, dict(objective=obj, gap=gap, step=step, device_ms=out.device_ms, sssp_ms=out.sssp_ms,
                             n_trees=out.n_trees, workspace_bytes=n.value)


def sssp_static(n_nodes, out_off, out_edge, edge_to, w, sources, pred, error=None, stream=None):
    """ts_sssp_static: shortest-path trees with no allocation anywhere (static device scratch, at most
    ts_sssp_static_max_nodes() nodes).  Every array is a CUDA torch tensor of 32-bit integers the caller
    owns (`pred`: n_sources * n_nodes words, output); enqueues one kernel on `stream` (default: current)."""
    import torch
    st = stream if stream is not None else torch.cuda.current_stream(pred.device)
    ptr = lambda t: None if t is None else t.data_ptr()
    _check(load().ts_sssp_static(int(n_nodes), int(out_edge.numel()), ptr(out_off), ptr(out_edge), ptr(edge_to),
                                 ptr(w), ptr(sources), int(sources.numel()), ptr(pred), ptr(error), st.cuda_stream))
