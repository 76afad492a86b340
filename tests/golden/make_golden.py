#!/usr/bin/env python
"""Writes tests/golden/trace_<cfg>.json by running ONLY the oracle (oracle/) on the seeded
workload of a BASELINE.json config, full length.

    python tests/golden/make_golden.py cfg1 cfg2 cfg3 cfg5 [--stride 600]
    python tests/golden/make_golden.py --emissions cfg1 cfg2 cfg5      # writes emissions_<cfg>.json

Stored per config (nothing here ever comes from the CUDA path):
  sha256     checksum of the generated input bundle (detects generator drift between machines)
  digests    the oracle's 64-bit state digest (SURVEY.md 8(d) "Parity") after steps
             stride, 2*stride, ..., and after the last step -- the sampled outputs the
             full-size GPU parity test compares against
  active     number of ACTIVE vehicles at the same steps
  counters   the oracle's work counters for the whole run: the cells a byte-scan method has to
             look at per vehicle-update, used by bench.py for the algorithmic bytes per update
  final      n_pending / n_active / n_arrived after the last step
  seconds    single-thread wall time of the oracle run (context only)
  edge_stats sums of the oracle's per-edge accumulators at the last mark (entered, exited,
             exit_steps_sum, sample_count_sum, sample_speedcode_sum, n_samples) and a position-weighted
             checksum of each: the digests do not cover these
  (--emissions: a separate file emissions_<cfg>.json with the whole-run totals of the section
             6.3.4 accumulators: per array the fp64 sum, the sum of the fp32 bit
             patterns and a position-weighted sum of the bit patterns, plus the final digest)
  final_state (written with the last mark) per array of the oracle's read_state -- status, edge, lane,
             route_idx, insert_step, arrive_step and the bit patterns of x and v, all V vehicles in id
             order -- its sum and a position-weighted checksum: what the digests (ACTIVE vehicles only) do
             not cover
  complete   false while the run is in progress: the file is rewritten after every stride, so an
             interrupted run of a very long config (config 4: 5.4e10 vehicle-updates, many hours of
             the single-threaded oracle) still leaves a usable prefix of digests
"""
import argparse
import json
import os
import sys
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
sys.path.insert(0, ROOT)

from oracle import Oracle                                    # noqa: E402
from paper_1807_01148_b200 import workload as W              # noqa: E402


def state_checksums(st):
    """Sum and position-weighted checksum of every per-vehicle array of a read_state() dict."""
    out = {}
    for k in ("status", "edge", "lane", "route_idx", "insert_step", "arrive_step", "x", "v"):
        a = np.asarray(st[k])
        u = (a.view(np.uint32) if a.dtype == np.float32 else a).astype(np.uint64)
        w = np.arange(1, len(u) + 1, dtype=np.uint64)
        out[k] = [int(u.sum()), int((u * w).sum() & np.uint64(0xFFFFFFFFFFFFFFFF))]
    return out


def run(name, stride, suffix="", threads=1):
    bundle = W.by_name(name)
    orc = Oracle(bundle)
    orc.set_threads(threads)
    steps = bundle["steps"]
    marks, digests, active = [], [], []
    sha = W.bundle_sha256(bundle)
    path = os.path.join(HERE, f"trace_{name}{suffix}.json")
    t0 = time.perf_counter()
    done = 0
    while done < steps:
        n = min(stride, steps - done)
        if n > 1:
            orc.step(n - 1)                      # only the digest at the mark is stored
        d = orc.step(1, digests=True)
        done += n
        marks.append(done)
        digests.append(f"{int(d[-1]):016x}")
        counts = orc.read_counts()
        active.append(int(counts["n_active"]))
        es = orc.read_edge_stats()
        w = np.arange(1, orc.E + 1, dtype=np.uint64)
        edge_stats = {k: [int(np.asarray(v, np.uint64).sum()), int((np.asarray(v, np.uint64) * w).sum() & np.uint64(0xFFFFFFFFFFFFFFFF))]
                      for k, v in es.items() if k != "n_samples"}
        edge_stats["n_samples"] = int(es["n_samples"])
        out = dict(name=bundle["name"], sha256=sha, steps=steps, stride=stride, complete=done == steps,
                   edge_stats=edge_stats,
                   marks=marks, digests=digests, active=active, counters=orc.counters(),
                   final=dict(n_pending=int(counts["n_pending"]), n_active=int(counts["n_active"]),
                              n_arrived=int(counts["n_arrived"])),
                   seconds=round(time.perf_counter() - t0, 1), threads=threads)
        if done == steps:
            out["final_state"] = state_checksums(orc.read_state())
        with open(path + ".tmp", "w") as f:
            json.dump(out, f, indent=1)
        os.replace(path + ".tmp", path)
    print(name, "->", path, f"{out['seconds']:.0f} s", out["counters"]["updates"], "updates", flush=True)


def _bits_checksums(a):
    u = np.asarray(a, np.float32).view(np.uint32).astype(np.uint64)
    w = np.arange(1, len(u) + 1, dtype=np.uint64)
    return dict(sum=float(np.asarray(a, np.float64).sum()), bits_sum=int(u.sum()),
                bits_weighted=int((u * w).sum() & np.uint64(0xFFFFFFFFFFFFFFFF)))


def run_emissions(name, stride, threads=1):
    bundle = W.by_name(name)
    sha = W.bundle_sha256(bundle)
    bundle = dict(bundle, params=dict(bundle["params"], emissions=1))
    orc = Oracle(bundle)
    orc.set_threads(threads)
    steps = bundle["steps"]
    t0 = time.perf_counter()
    done, last = 0, None
    while done < steps:
        n = min(stride, steps - done)
        if n > 1:
            orc.step(n - 1)
        last = orc.step(1, digests=True)[-1]
        done += n
    em = orc.read_emissions()
    out = dict(name=bundle["name"], sha256=sha, steps=steps, final_digest=f"{int(last):016x}",
               updates=orc.counters()["updates"], co_g=_bits_checksums(em["co_g"]),
               fuel_ml=_bits_checksums(em["fuel_ml"]), seconds=round(time.perf_counter() - t0, 1),
               threads=threads)
    path = os.path.join(HERE, f"emissions_{name}.json")
    with open(path, "w") as f:
        json.dump(out, f, indent=1)
    print(name, "->", path, f"{out['seconds']:.0f} s", flush=True)


if __name__ == "__main__":
    ap = argparse.ArgumentParser()
    ap.add_argument("configs", nargs="+")
    ap.add_argument("--stride", type=int, default=600)
    ap.add_argument("--suffix", default="", help="write trace_<cfg><suffix>.json (a second, incremental run beside a long one)")
    ap.add_argument("--emissions", action="store_true", help="write emissions_<cfg>.json instead of a trace")
    ap.add_argument("--threads", type=int, default=1,
                    help="host threads for the oracle's intent loop (orc_set_threads; results do not depend on it)")
    a = ap.parse_args()
    for c in a.configs:
        if a.emissions:
            run_emissions(c, a.stride, a.threads)
        else:
            run(c, a.stride, a.suffix, a.threads)
