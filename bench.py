#!/usr/bin/env python
"""bench.py -- vehicle-updates/s of the traffic microsimulation on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg3] [--impl reference]

A bench "step" is ONE complete simulated run of the workload (ts_reset, then every simulation
step of the config through ts_step): one pass of the whole hot path (SURVEY.md 8(a) rows
A1-A11) over one batch of synthetic input.  One vehicle-update = one ACTIVE vehicle advanced
one simulation step.  `value` is measured with the inputs resident in HBM (CUDA events on the
launching stream around ts_step); `e2e` goes through the C ABI with host buffers: ts_create
(validation + H2D of network, routes, departures), ts_step, ts_read_state (D2H).

Multi-GPU: the path does not shard -- replicas only.  Under torchrun every
rank runs an independent replica of the same workload; no data-path collective exists.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "vehicle_updates_per_sec"
UNIT = "vehicle-updates/s"

# Algorithmic bytes per vehicle-update:
#   32 (state read) + 8 (x, v written) + S_own + S_lc + 2 (atlas erase + store)
# with S_own / S_lc = mean atlas cells scanned per update in the own lane (+ next edge) and in
# the lane-change target lane, taken from the oracle's work counters in the stored trace of the
# config (tests/golden/trace_<cfg>[_partial].json, written by tests/golden/make_golden.py): the
# whole run where the oracle has finished it, else the prefix it has reached -- the JSON line says
# which in roofline.bytes_source, and the figure moves with the prefix (cells scanned per update
# fall as traffic builds up).
SCAN_CELLS_FALLBACK = {"cfg1": 87.3 + 12.9, "cfg2": 11.4 + 2.7, "cfg3": 60.0, "cfg5": 30.0}


def load_workload(name):
    from paper_1807_01148_b200 import workload as W
    try:
        return W.by_name(name)
    except KeyError as e:
        raise SystemExit(str(e))


def measured_traffic(name, geometry):
    """DRAM bytes (dram__bytes_read.sum + dram__bytes_write.sum) of the step kernel over one whole
    run of workload `name`, from the committed ncu capture of every launch of the geometry the
    bench line was measured with (the same two metrics a --set full capture holds; one launch of it is
    captured in full beside it) (profiles/r02e_kernel_traffic.csv:
    workload,geometry,dram_read_bytes,dram_write_bytes,launches; geometry = "adaptive" -- the default:
    the sum over the launches of every 2048-step chunk -- or "threadsNNN").  None if that geometry
    was not captured: a number from another geometry is not this run's traffic."""
    path = os.path.join(ROOT, "profiles", "r02e_kernel_traffic.csv")
    try:
        for line in open(path):
            f = [t.strip() for t in line.split(",")]
            if len(f) >= 4 and f[0] == name and f[1] == geometry:
                return float(f[2]) + float(f[3])
    except OSError:
        pass
    return None


def load_trace(name):
    for suffix in ("", "_partial"):
        try:
            return json.load(open(os.path.join(ROOT, "tests", "golden", f"trace_{name}{suffix}.json")))
        except (OSError, ValueError):
            continue
    return None


def bytes_per_update(name):
    """32 + 8 + scanned cells + 2 (see the comment above); cells from the oracle's counters.
    Returns (bytes, cells, source, bytes with every scan rounded up to 16-cell pieces, its source)."""
    t = load_trace(name)
    try:
        c = t["counters"]
        cells = (c["own_cells"] + c["next_cells"] + c["lc_cells"]) / c["updates"]
        what = "full run" if t.get("complete", True) else f"first {t['marks'][-1]} of {t['steps']} steps"
        if "own_chunks16" in c:
            cells16 = 16.0 * (c["own_chunks16"] + c["next_chunks16"] + c["lc_chunks16"]) / c["updates"]
            src16 = "oracle counters (every scan rounded up to 16 cells)"
        else:       # trace written before the oracle counted pieces: half a piece per scan on average
            scans = (c["updates"] + 2 * c["lc_evals"]) / c["updates"] + min(1.0, c["next_cells"] / max(1, c["own_cells"]))
            cells16, src16 = cells + 7.5 * scans, "estimate: raw cells + 7.5 per scan"
        return 32 + 8 + cells + 2, cells, f"oracle counters, {what}", 32 + 8 + cells16 + 2, src16
    except (TypeError, KeyError, ZeroDivisionError):
        cells = SCAN_CELLS_FALLBACK.get(name.replace("_small", ""), 60.0)
        return 32 + 8 + cells + 2, cells, "estimate", 32 + 8 + cells + 7.5 + 2, "estimate"


class ClockSampler:
    """nvidia-smi clocks and throttle reasons DURING the timed region (B200_PROFILING.md)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "100"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._pump, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _pump(self):
        for line in self.proc.stdout:
            self.rows.append(line.strip())

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        self.thread.join(timeout=2)
        sm, mx, reasons = [], None, set()
        for r in self.rows:
            f = [t.strip() for t in r.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx = float(f[1])
            except ValueError:
                continue
            for name, val in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), f[3:7]):
                if val.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": mx,
                "reasons": sorted(reasons), "samples": len(sm)}


def time_oracle(bundle, budget_s, chunk=600):
    """The oracle as it stands, one thread, on a bounded prefix of the workload."""
    from oracle import Oracle
    orc = Oracle(bundle)
    t0 = time.perf_counter()
    steps = 0
    while steps < bundle["steps"]:
        n = min(chunk, bundle["steps"] - steps)
        orc.step(n)
        steps += n
        if time.perf_counter() - t0 > budget_s:
            break
    dt = time.perf_counter() - t0
    upd = orc.counters()["updates"]
    orc.close()
    return upd, dt, steps


def whole_run_baseline(name):
    """The oracle's rate over the WHOLE run of the config, from the stored trace's wall time (written
    by tests/golden/make_golden.py on the build machine, not on this box): context for the prefix
    sample timed here, which covers only the free-flowing start of the run."""
    t = load_trace(name)
    if not t or not t.get("seconds") or not t.get("complete", True):
        return {"whole_run_value": None}
    return {"whole_run_value": t["counters"]["updates"] / t["seconds"], "whole_run_threads": t.get("threads", 1),
            "whole_run_note": "stored trace (tests/golden), oracle wall time on the machine that wrote it"}


def whole_job(total_ms_local, units_per_rank, dist=None, device="cpu"):
    """Replicas only: every rank ran the same number of units; the job's time
    is the MAX over ranks, its work the sum.  Returns (units/s of the whole job, max ms)."""
    import torch
    t = torch.tensor([float(total_ms_local)], dtype=torch.float64, device=device)
    world = 1
    if dist is not None:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        world = dist.get_world_size()
    ms = float(t.item())
    return units_per_rank * world / (ms / 1e3), ms


def run_reference(args):
    """--impl reference: the oracle on the host cores (rank 0 only)."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    bundle = load_workload(args.workload)
    budget = max(2.0, min(20.0, 150.0 / max(1, args.steps + args.warmup)))
    times, upds, steps = [], [], 0
    for i in range(args.warmup + args.steps):
        upd, dt, steps = time_oracle(bundle, budget)
        if i >= args.warmup:
            times.append(dt); upds.append(upd)
    value = sum(upds) / sum(times)
    sample = f"first {steps} of {bundle['steps']} simulation steps of {bundle['name']} ({upds[-1]} vehicle-updates) per bench step"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * sum(times) / len(times),
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
        "data": "synthetic", "config": {"workload": bundle["name"], "sample": sample},
        "cpu_baseline": dict({"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample,
                              "box_cores": os.cpu_count()}, **whole_run_baseline(args.workload)),
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


def run_reroute(args):
    """--reroute: the paper's assignment loop: simulate, measure, re-route all / all /
    half / a quarter of the vehicles, four times; one bench "step" is the whole loop.  Prints the
    usual line (vehicle-updates/s over the loop, ts_reroute included) plus a `reroute` object with
    the per-iteration gap between the times the routes were chosen with and the times simulated,
    and a roofline object for the shortest-path kernel."""
    import torch
    import paper_1807_01148_b200 as pkg
    from paper_1807_01148_b200 import workload as W
    torch.cuda.set_device(0)
    bundle = load_workload(args.workload)
    cap = int(len(bundle["route_edges"]) * 2 + 1024)
    b = dict(bundle, params=dict(bundle["params"], route_capacity=cap))
    sim = pkg.Sim(b, "cuda:0")
    stream = torch.cuda.current_stream()
    wf = W.free_flow_weights(b)
    steps = args.sim_steps or b["steps"]
    E, dt = b["n_edges"], b["params"]["dt"]
    rows, ms_all, updates_all, launches = [], [], [], 0
    sampler = ClockSampler(0)
    for rep_ in range(args.warmup + args.steps):
        if rep_ == args.warmup:
            sampler.start()
        if rep_:                                        # every repetition starts from the routes given
            sim.close()
            sim = pkg.Sim(b, "cuda:0")
        used = wf.astype(np.float64) / W.W_UNIT          # weights the routes in use were chosen with, in steps
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        e0.record(stream)
        upd, rows = 0, []
        for it in range(4):
            sim.step(steps)
            st = sim.read_counts()
            upd += int(st["vehicle_updates"])
            es = sim.read_edge_stats()
            seen = es["exited"] > 0
            sim_t = es["exit_steps_sum"][seen] / es["exited"][seen]
            t_host = time.perf_counter()
            info = sim.reroute(wf, W.reroute_mask(b["n_vehicles"], it))
            host_ms = 1e3 * (time.perf_counter() - t_host)
            rows.append({"iteration": it, "n_rerouted": info["n_rerouted"], "n_trees": info["n_trees"],
                         "sssp_ms": info["sssp_ms"], "device_ms": info["device_ms"], "call_ms": host_ms,
                         "arrived": int(st["n_arrived"]), "edges_with_exits": int(seen.sum()),
                         "mean_abs_gap_s": float(np.abs(used[seen] - sim_t).mean() * dt),
                         "mean_simulated_s": float(sim_t.mean() * dt)})
            used = info["w"].astype(np.float64) / W.W_UNIT
        e1.record(stream)
        torch.cuda.synchronize()
        if rep_ >= args.warmup:
            ms_all.append(e0.elapsed_time(e1)); updates_all.append(upd)
            launches += 4 * (2 * ((steps + 2047) // 2048) + 9)
    clocks = sampler.stop()
    sim.close()
    peaks_path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    peak = float(json.load(open(peaks_path))["hbm_gbs"]) if os.path.exists(peaks_path) else 6650.0
    trees = sum(r["n_trees"] for r in rows)
    sssp_s = sum(r["sssp_ms"] for r in rows) / 1e3
    # per tree every edge is relaxed at least once: label of the tail (8 B), out_edge + edge_to + weight
    # (12 B), label of the head read and written by the atomicMin (16 B)
    alg = 36.0 * E * trees
    value = sum(updates_all) / (sum(ms_all) / 1e3)
    print(json.dumps({
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": 1, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": sum(ms_all) / len(ms_all), "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32 (traffic), u32/u64 (routing weights and labels)", "data": "synthetic",
        "config": {"workload": bundle["name"] + " + 4 re-routing iterations (PAPER.md:386)", "vehicles": b["n_vehicles"],
                   "edges": E, "sim_steps_per_iteration": steps},
        "reroute": rows, "gpu_launches": launches, "clocks": clocks,
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": int(4 * (E * 4 + b["n_vehicles"])),
                "d2h_bytes_per_step": int(4 * (E * 28 + b["n_vehicles"] * 16)),
                "note": "the loop is driven through the C ABI: statistics D2H, masks and free-flow weights H2D, "
                        "the departure-queue index rebuilt on the host inside ts_reroute"},
        "roofline": {"bound": "hbm", "kernel": "k_rr_sssp", "achieved": alg / sssp_s / 1e9 if sssp_s else None, "peak": peak,
                     "unit": "GB/s", "frac": alg / sssp_s / 1e9 / peak if sssp_s else None, "traffic": None,
                     "bytes_per_unit": 36.0, "unit_of_work": "edge relaxation (one per edge per tree at least)",
                     "trees": trees, "kernel_ms_total": 1e3 * sssp_s},
    }))


def run_sue(args):
    """--sue: the paper's static traffic assignment (Frank-Wolfe with BPR times) on the
    workload's network and OD demand (workload.sue_inputs), SURVEY.md 8(f) row 5.  One bench "step" is one
    ts_sue_solve call from host buffers.  The usual line with metric = shortest-path trees per second (the
    dominant kernel is the tree kernel shared with ts_reroute), its roofline object and the convergence."""
    import torch
    import paper_1807_01148_b200 as pkg
    from paper_1807_01148_b200 import workload as W
    torch.cuda.set_device(0)
    bundle = load_workload(args.workload)
    inp = W.sue_inputs(bundle, horizon_s=args.sue_horizon)
    a = (bundle["n_nodes"], bundle["edge_from"], bundle["edge_to"], inp["t0"], inp["cap"], inp["od_origin"],
         inp["od_dest"], inp["od_trips"])
    ms, info = [], None
    sampler = ClockSampler(0)
    for rep_ in range(args.warmup + args.steps):
        if rep_ == args.warmup:
            sampler.start()
        t0 = time.perf_counter()
        flow, times, info = pkg.sue_solve(*a, iterations=args.sue_iterations)
        if rep_ >= args.warmup:
            ms.append(1e3 * (time.perf_counter() - t0))
    clocks = sampler.stop()
    peaks_path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    peak = float(json.load(open(peaks_path))["hbm_gbs"]) if os.path.exists(peaks_path) else 6650.0
    E, trees = bundle["n_edges"], int(info["n_trees"])
    alg = 36.0 * E * trees
    sssp_s = info["sssp_ms"] / 1e3
    print(json.dumps({
        "metric": "shortest_path_trees_per_sec", "value": trees * len(ms) / (sum(ms) / 1e3), "unit": "trees/s", "n_gpus": 1,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": sum(ms) / len(ms), "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64 (flows, times), u32/u64 (weights, labels, all-or-nothing flows)",
        "data": "synthetic",
        "config": {"workload": bundle["name"] + " static user equilibrium (PAPER.md:307-338)", "nodes": bundle["n_nodes"],
                   "edges": E, "od_pairs": int(len(inp["od_trips"])), "trips": int(inp["od_trips"].sum()),
                   "origins": int(len(np.unique(inp["od_origin"]))), "iterations": args.sue_iterations,
                   "demand_horizon_s": args.sue_horizon, "workspace_bytes": int(info["workspace_bytes"])},
        "sue": {"relative_gap": [float(g) for g in info["gap"]], "step": [float(x) for x in info["step"]],
                "objective_first_last": [float(info["objective"][0]), float(info["objective"][-1])],
                "device_ms": float(info["device_ms"]), "tree_kernel_ms": float(info["sssp_ms"]),
                "max_v_over_c": float((flow / inp["cap"]).max())},
        "e2e": {"value": trees * len(ms) / (sum(ms) / 1e3), "unit": "trees/s",
                "h2d_bytes_per_step": int(E * 24 + len(inp["od_trips"]) * 16), "d2h_bytes_per_step": int(E * 16),
                "note": "the timed call takes host buffers and returns host arrays"},
        "gpu_launches": len(ms) * (args.sue_iterations + 1) * 50, "clocks": clocks,
        "roofline": {"bound": "hbm", "kernel": "k_rr_sssp", "achieved": alg / sssp_s / 1e9, "peak": peak, "unit": "GB/s",
                     "frac": alg / sssp_s / 1e9 / peak, "traffic": None, "bytes_per_unit": 36.0,
                     "unit_of_work": "edge relaxation (one per edge per tree at least)", "trees": trees},
    }))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="cfg3")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--mode", type=int, default=1, help="1 persistent kernel (default), 0 two launches per step")
    ap.add_argument("--sim-steps", type=int, default=0, help="override the config's simulation steps (diagnostics)")
    ap.add_argument("--start-step", type=int, default=0,
                    help="advance this many simulation steps untimed before the timed window (diagnostics)")
    ap.add_argument("--threads", type=int, default=0, help="CTA size of the persistent kernel (tuning)")
    ap.add_argument("--blocks-per-sm", type=int, default=0)
    ap.add_argument("--sort-period", type=int, default=-1, help="steps between compaction + re-sort (tuning)")
    ap.add_argument("--opt", action="append", default=[], metavar="KEY=VALUE",
                    help="ts_set_option(KEY, VALUE) before the run (tuning knobs; results never depend on them)")
    ap.add_argument("--profile", action="store_true", help="clock the phases inside the persistent kernel")
    ap.add_argument("--emissions", action="store_true",
                    help="keep the per-vehicle CO / fuel totals of PAPER.md:408-423 (SURVEY.md 8(f) row 2) during the run")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true", help="skip the end-to-end leg (profiling runs)")
    ap.add_argument("--no-window", action="store_true", help="skip the busiest-window pass (profiling runs)")
    ap.add_argument("--reroute", action="store_true",
                    help="the four-iteration re-routing loop of PAPER.md:386 on the workload (SURVEY.md 8(f) row 1)")
    ap.add_argument("--sue", action="store_true",
                    help="static user equilibrium by Frank-Wolfe + BPR on the workload's network and demand (SURVEY.md 8(f) row 5)")
    ap.add_argument("--sue-iterations", type=int, default=10)
    ap.add_argument("--sue-horizon", type=float, default=3600.0, help="seconds over which the trips are spread (demand rate)")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    if args.reroute:
        return run_reroute(args)
    if args.sue:
        return run_sue(args)
    if args.warmup < 3:
        print("note: timing rules ask for >= 3 warm-up steps", file=sys.stderr)

    import torch
    import paper_1807_01148_b200 as pkg

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product has no CPU fallback")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    bundle = load_workload(args.workload)
    if args.emissions:
        bundle = dict(bundle, params=dict(bundle["params"], emissions=1))
    sim_steps = args.sim_steps or (bundle["steps"] - args.start_step)
    stream = torch.cuda.current_stream()
    sim = pkg.Sim(bundle, f"cuda:{local}", mode=args.mode)
    tuning = {}
    if args.threads:
        tuning["threads"] = args.threads
    if args.blocks_per_sm:
        tuning["blocks_per_sm"] = args.blocks_per_sm
    if args.sort_period >= 0:
        tuning["sort_period"] = args.sort_period
    if args.profile:
        tuning["profile"] = 1
    for kv in args.opt:
        key, _, val = kv.partition("=")
        tuning[key] = int(val)
    for key, val in tuning.items():
        sim.set_option(key, val)

    flush = torch.empty(256 << 20, dtype=torch.uint8, device=f"cuda:{local}")   # > 126 MB L2

    def one_run():
        sim.reset()
        if args.start_step:
            sim.set_option("mode", 1)                    # one persistent launch to get there
            sim.step(args.start_step)                    # untimed: reach the window of interest
            sim.set_option("mode", args.mode)
            base = int(sim.read_counts()["vehicle_updates"])
        else:
            base = 0
        flush.fill_(1)                                   # L2 flush between timed iterations
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        sim.step(sim_steps)                              # the whole hot path, device-resident inputs
        e1.record(stream)
        return e0, e1, base

    for _ in range(args.warmup):
        one_run()
    barrier()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    evs = [one_run() for _ in range(args.steps)]
    barrier()
    clocks = sampler.stop() if rank == 0 else None
    ms = [a.elapsed_time(b) for a, b, _ in evs]
    counts = sim.read_counts()
    phase_ns = sim.read_profile() if args.profile else None
    updates = int(counts["vehicle_updates"]) - evs[-1][2]   # per timed window (reset zeroes the counter)
    value, total_ms = whole_job(sum(ms), updates * args.steps, dist, f"cuda:{local}")

    # end to end through the C ABI with host buffers (pinned where torch can pin them)
    h2d = sum(int(np.asarray(bundle[k]).nbytes) for k in (
        "edge_from", "edge_to", "edge_len_m", "edge_lanes", "edge_vlim", "node_ctrl", "sig_green_steps",
        "sig_allred_steps", "sig_offset_steps", "route_off", "route_edges", "depart_time_s", "v0_mult", "mand_dist_m"))
    V = bundle["n_vehicles"]
    d2h = V * (1 + 4 + 1 + 4 + 4 + 4 + 4 + 4 + 4) + 64
    # the rate over the 3600-step window with the most active vehicles, beside the whole run
    window = None
    if rank == 0 and not args.start_step and sim_steps > 3600 and not args.no_window:
        sim.reset()
        prev, best = 0, None
        for w0 in range(0, sim_steps, 3600):
            n = min(3600, sim_steps - w0)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream); sim.step(n); e1.record(stream)
            tot = int(sim.read_counts()["vehicle_updates"])
            if n == 3600 and (best is None or tot - prev > best[1]):
                best = (w0, tot - prev, e0.elapsed_time(e1))
            prev = tot
        if best:
            window = {"first_step": best[0], "steps": 3600, "vehicle_updates": best[1], "mean_active": best[1] / 3600,
                      "value": best[1] / (best[2] / 1e3), "unit": UNIT, "us_per_sim_step": 1e3 * best[2] / 3600}
    sim.close()
    del sim
    pinned = dict(bundle)
    for k in ("route_edges", "route_off", "depart_time_s", "v0_mult", "mand_dist_m"):
        t = torch.from_numpy(np.ascontiguousarray(bundle[k]).view(np.uint8)).pin_memory()
        pinned[k] = t.numpy().view(bundle[k].dtype)
        pinned["_keep_" + k] = t
    e2e_ms = []
    for i in range(0 if (args.start_step or args.no_e2e) else 1 + max(1, args.steps)):   # diagnostics have no e2e leg
        barrier()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        s2 = pkg.Sim(pinned, f"cuda:{local}", mode=args.mode)     # ts_query_workspace + ts_create: H2D
        for key, val in tuning.items():
            s2.set_option(key, val)
        s2.step(sim_steps)
        st = s2.read_state()                                       # D2H of the whole state
        e1.record(stream)
        torch.cuda.synchronize()
        if i > 0:
            e2e_ms.append(e0.elapsed_time(e1))
        assert int(st["vehicle_updates"]) == updates
        s2.close()
    e2e_value = whole_job(sum(e2e_ms), updates * len(e2e_ms), dist, f"cuda:{local}")[0] if e2e_ms else None

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    peaks_path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(peaks_path):
        peak, peak_src = float(json.load(open(peaks_path))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    else:
        peak, peak_src = 6650.0, "fallback (B200_PROFILING.md)"
    bpu, cells, bsrc, bpu16, bsrc16 = bytes_per_update(args.workload)
    launch_s = (sum(ms) / len(ms)) / 1e3                  # one k_persistent launch per bench step
    achieved = bpu * updates / launch_s / 1e9
    # mode 1: one cooperative launch per ts_step call, or -- adaptive CTA size, the default when no
    # geometry is asked for -- two per chunk of 2048 steps, of which the device runs one
    adaptive = args.mode == 1 and not (args.threads or args.blocks_per_sm or args.profile)
    launches_per_run = (2 * sim_steps if args.mode != 1 else
                        2 * ((sim_steps + 2047) // 2048) if adaptive else 1)
    geometry = "adaptive" if adaptive else f"threads{args.threads or 640}"
    traffic = (measured_traffic(args.workload, geometry)
               if args.mode == 1 and not args.start_step and not args.sim_steps and not args.emissions else None)
    traffic_src = (f"ncu dram__bytes_read.sum + dram__bytes_write.sum, every launch of one whole run, geometry {geometry} (profiles/r02e_kernel_traffic.csv)" if traffic is not None
                   else f"no ncu capture of geometry {geometry} for this workload")
    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": total_ms / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
        "data": "synthetic",
        "config": {"workload": bundle["name"], "vehicles": V, "edges": bundle["n_edges"],
                   "sim_steps_per_bench_step": sim_steps, "vehicle_updates_per_bench_step": updates,
                   "start_step": args.start_step, "tuning": tuning, "emissions": bool(args.emissions), "phase_ns_per_sim_step": phase_ns,
                   "parallelism": "replicas only" if world > 1 else "single GPU",
                   "step_kernel": ("persistent cooperative, CTA size chosen on the device per 2048 steps (640 / 768 threads)" if adaptive
                                   else "persistent cooperative" if args.mode == 1 else "two launches per sim step"),
                   "l2": "flushed between timed iterations (256 MiB fill) and inputs (routes+atlas) exceed L2"},
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                "ms_per_step": sum(e2e_ms) / len(e2e_ms) if e2e_ms else None},
        "gpu_launches": args.steps * launches_per_run,
        "clocks": clocks,
        "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s",
                     "frac": achieved / peak, "frac_nominal": achieved / 8000.0, "peak_nominal": 8000.0,
                     "traffic": traffic, "traffic_source": traffic_src,
                     "bytes_per_update_chunk16": bpu16, "achieved_chunk16": bpu16 * updates / launch_s / 1e9,
                     "frac_chunk16": bpu16 * updates / launch_s / 1e9 / peak, "chunk16_source": bsrc16,
                     "busiest_window": window,
                     "peak_source": peak_src,
                     "kernel": "k_persistent" if args.mode == 1 else "k_phase1+k_phase2",
                     "bytes_per_update": bpu, "scan_cells_per_update": cells, "bytes_source": bsrc,
                     "us_per_sim_step": 1e6 * launch_s / sim_steps},
    }
    if not args.no_cpu_baseline:
        upd, dt, steps = time_oracle(bundle, 15.0)
        out["cpu_baseline"] = {"value": upd / dt, "unit": UNIT, "cores": 1, "kind": "oracle",
                               "box_cores": os.cpu_count(),
                               "sample": f"first {steps} of {bundle['steps']} simulation steps of {bundle['name']} "
                                         f"({upd} vehicle-updates, {dt:.1f} s, single thread): the free-flowing "
                                         "start of the run, where the oracle is fastest"}
        out["cpu_baseline"].update(whole_run_baseline(args.workload))
    print(json.dumps(out))
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
