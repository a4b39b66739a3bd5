#!/usr/bin/env python
"""bench.py — throughput of the skeleton hot path on B200 (contract: see DESIGN.md "Measurement").

One *step* = one pass of the whole hot path over one batch of synthetic input: every skeleton of
SURVEY.md §8(a) at the largest size BASELINE.json's configs give it (Map saxpy 2^26, int32 Reduce
sum+max 2^26, MapReduce dot 2^26, MapOverlap 1D r in {1,4,16} x {constant-0, duplicate} 2^26,
MapOverlap 2D 5x5 / 9x9 and the separable r=8 row+column pair on 8192^2, int32 Scan inclusive +
exclusive 2^28). `value` = algorithmic bytes of the step / device time of the step (GB/s), inputs
resident in HBM. `e2e` = the same through host buffers (uploads and downloads inside the timed
region). Every working set is > L2 (126 MB), so no flush is needed between iterations.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--scale S] [--impl reference]

N > 1 (under torchrun): independent replicas, one per GPU ("replicas only": the path does not
shard, BASELINE.json L5). --impl reference times the CPU oracle (the only reference this tier has).
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

# dram__bytes_read.sum + dram__bytes_write.sum per launch at full size, per kernel VARIANT, from the `ncu --set full`
# captures listed in profiles/r02_ncu_traffic.csv (command: profiles/r02_ncu_traffic.md). A variant that has no row
# there reports "traffic": null instead of a stale number.
TRAFFIC_CSV = os.path.join(ROOT, "profiles", "r02_ncu_traffic.csv")


def ncu_traffic(op_name: str, variant: str):
    if not os.path.exists(TRAFFIC_CSV):
        return None
    import csv
    with open(TRAFFIC_CSV) as f:
        for row in csv.DictReader(f):
            if row["bench_op"] == op_name and row["variant"] == variant:
                return int(float(row["dram_bytes_read"]) + float(row["dram_bytes_write"]))
    return None

METRIC = "skeleton throughput (algorithmic GB/s over one pass of all skeletons at their largest config)"
UNIT = "GB/s"


def log(*a):
    print(*a, file=sys.stderr, flush=True)


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            return json.load(f).get("hbm_gbs", 6650.0), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md: 6.65 TB/s)"


# --------------------------------------------------------------------------------------------------
def sizes(scale: float):
    lg = lambda full: max(12, int(round(full + np.log2(scale))))  # noqa: E731
    side = 1 << max(6, int(round(13 + np.log2(scale) / 2)))
    return {"n26": 1 << lg(26), "n28": 1 << lg(28), "side": side}


def gen_inputs(sz):
    import skel_inputs as I
    t = time.time()
    d = {
        "x": I.uniform_pm1_f32(I.config_seed(2, 0), sz["n26"]),
        "y": I.uniform_pm1_f32(I.config_seed(2, 1), sz["n26"]),
        "vi": I.uniform_int_i32(I.config_seed(2, 2), sz["n26"], 1000),
        "s": I.uniform01_f32(I.config_seed(3, 0), sz["n26"]),
        "X": I.uniform01_f32(I.config_seed(4, 0), sz["side"] * sz["side"]).reshape(sz["side"], sz["side"]),
        "scan": I.uniform_int_i32(I.config_seed(5, 0), sz["n28"], 15),
        "w": {r: I.positive_weights_f32(I.config_seed(3, 10 + r), 2 * r + 1) for r in (1, 4, 8, 16)},
        "W5": I.positive_weights_f32(I.config_seed(4, 1), 25),
        "W9": I.positive_weights_f32(I.config_seed(4, 2), 81),
        "wr8": I.positive_weights_f32(I.config_seed(4, 3), 17),
        "wc8": I.positive_weights_f32(I.config_seed(4, 4), 17),
    }
    log(f"[bench] inputs generated in {time.time() - t:.1f} s")
    return d


class Workload:
    """Containers + the ordered list of skeleton calls of one step."""

    def __init__(self, S, ctx, d, sz):
        self.S, self.ctx, self.sz = S, ctx, sz
        n26, n28, side = sz["n26"], sz["n28"], sz["side"]
        self.vx, self.vy = ctx.vector_from(d["x"]), ctx.vector_from(d["y"])
        self.vr = ctx.vector(n26)
        self.vi = ctx.vector_from(d["vi"])
        self.vs, self.vso = ctx.vector_from(d["s"]), ctx.vector(n26)
        self.mX, self.mT, self.mO = ctx.matrix_from(d["X"]), ctx.matrix(side, side), ctx.matrix(side, side)
        self.vscan, self.vscan_o = ctx.vector_from(d["scan"]), ctx.vector(n28, S.I32)
        self.res = ctx.vector(8, S.I32)
        self.resf = ctx.vector(8, S.F32)
        self.inputs = [self.vx, self.vy, self.vi, self.vs, self.mX, self.vscan]
        self.outputs = [self.vr, self.vso, self.mO, self.vscan_o, self.res, self.resf]
        m = side * side
        ops = []
        add = lambda name, fam, fn, nbytes, elems: ops.append((name, fam, fn, nbytes, elems))  # noqa: E731
        # the Scan goes first: its 1 GiB result is the largest download of the end-to-end step and, prefetched, overlaps
        # the uploads of everything that follows (the order of the 16 calls does not matter to the device-resident numbers)
        add("scan_inclusive_i32", "scan", lambda: ctx.scan(S.FN_ADD, S.SCAN_INCLUSIVE, 0, self.vscan, self.vscan_o), 8 * n28, n28)
        add("scan_exclusive_i32", "scan", lambda: ctx.scan(S.FN_ADD, S.SCAN_EXCLUSIVE, 0, self.vscan, self.vscan_o), 8 * n28, n28)
        add("map_saxpy_f32", "map", lambda: ctx.map(S.FN_SAXPY, 2.5, self.vx, self.vy, self.vr), 12 * n26, n26)
        # the dot product (read-only, 512 MB) runs between saxpy and the two Reduce calls: whatever follows saxpy is timed
        # while the 256 MB that saxpy left dirty in L2 are written back, and a 268 MB Reduce is the call that shows it most
        add("mapreduce_dot_f32", "mapreduce",
            lambda: ctx.mapreduce_to(S.FN_MULT, S.FN_ADD, 0.0, self.vx, self.vy, self.resf, 0), 8 * n26, n26)
        add("reduce_sum_i32", "reduce", lambda: ctx.reduce_to(S.FN_ADD, self.vi, self.res, 0), 4 * n26, n26)
        add("reduce_max_i32", "reduce", lambda: ctx.reduce_to(S.FN_MAX, self.vi, self.res, 1), 4 * n26, n26)
        for r in (1, 4, 16):
            for edge, en in ((S.EDGE_CONSTANT, "const0"), (S.EDGE_DUPLICATE, "dup")):
                add(f"overlap1d_r{r}_{en}", "overlap1d",
                    (lambda r=r, edge=edge: ctx.mapoverlap_1d(d["w"][r], r, edge, 0.0, self.vs, self.vso)), 8 * n26, n26)
        add("overlap2d_5x5_dup", "overlap2d", lambda: ctx.mapoverlap_2d(d["W5"], 2, 2, S.EDGE_DUPLICATE, 0.0, self.mX, self.mO), 8 * m, m)
        add("overlap2d_9x9_dup", "overlap2d", lambda: ctx.mapoverlap_2d(d["W9"], 4, 4, S.EDGE_DUPLICATE, 0.0, self.mX, self.mO), 8 * m, m)
        add("overlap1d_rows_r8_dup", "overlap1d",
            lambda: ctx.mapoverlap_1d_matrix(d["wr8"], 8, S.EDGE_DUPLICATE, 0.0, S.AXIS_ROW, self.mX, self.mT), 8 * m, m)
        add("overlap1d_cols_r8_dup", "overlap1d_col",
            lambda: ctx.mapoverlap_1d_matrix(d["wc8"], 8, S.EDGE_DUPLICATE, 0.0, S.AXIS_COL, self.mT, self.mO), 8 * m, m)
        self.ops = ops
        # e2e: which outputs are final after which call of the step (skel_*_prefetch_host right there)
        self.last_writer = {"map_saxpy_f32": [self.vr], "reduce_max_i32": [self.res, self.resf],
                            "overlap1d_r16_dup": [self.vso], "overlap1d_cols_r8_dup": [self.mO],
                            "scan_exclusive_i32": [self.vscan_o]}
        self.bytes_per_step = sum(o[3] for o in ops)
        self.elems_per_step = sum(o[4] for o in ops)

    def step(self, events=None, prefetch=False):
        import torch
        for i, (name, _, fn, _, _) in enumerate(self.ops):
            if events is not None:
                events[i][0].record()
            fn()
            if events is not None:
                events[i][1].record()
            if prefetch and name in self.last_writer:  # the output is final: start its download now (copy stream)
                for c in self.last_writer[name]:
                    c.prefetch_host()

    def e2e_step(self, prefetch=True):
        """Host produces new inputs (pinned buffers), all skeletons run, host reads every output. prefetch: every
        output starts its download (skel_*_prefetch_host, copy stream) as soon as the call that finishes it is
        enqueued, so downloads overlap the uploads and kernels of the later calls (PCIe is full duplex)."""
        S = self.S
        for c in self.inputs:  # host write access: the device copy becomes stale -> next use uploads
            c.host_view(S.WRITE)
            c.release()
        self.step(prefetch=prefetch)
        tot = 0.0
        for c in self.outputs:  # host read access: downloads
            v = c.host_view(S.READ)
            tot += float(v.reshape(-1)[0])
            c.release()
        return tot

    def verify(self, d):
        """Cheap O(n) property checks on the step's outputs (full parity lives in tests/)."""
        S = self.S
        res = self.res.numpy()
        assert int(res[0]) & 0xFFFFFFFF == int(d["vi"].astype(np.int64).sum()) & 0xFFFFFFFF, "reduce sum mismatch"
        assert int(res[1]) == int(d["vi"].max()), "reduce max mismatch"
        dot = float(self.resf.numpy()[0])
        ref = float(np.dot(d["x"].astype(np.float64), d["y"].astype(np.float64)))
        assert abs(dot - ref) <= 1e-5 * float(np.abs(d["x"].astype(np.float64) * d["y"]).sum()), "dot mismatch"
        sc = self.vscan_o.numpy()  # last call of the step was the exclusive scan
        x = d["scan"]
        assert sc[0] == 0 and np.array_equal(sc[1:] - sc[:-1], x[:-1]), "scan mismatch"
        r = self.vr.numpy()
        assert np.array_equal(r[:4096], (np.float32(2.5) * d["x"][:4096].astype(np.float64) + d["y"][:4096]).astype(np.float32)) or \
            np.max(np.abs(r[:4096] - (2.5 * d["x"][:4096].astype(np.float64) + d["y"][:4096]))) < 1e-6, "map mismatch"

    def destroy(self):
        for c in self.inputs + self.outputs + [self.mT]:
            c.destroy()


# --------------------------------------------------------------------------------------------------
class ClockSampler:
    Q = "clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown," \
        "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"

    def __init__(self, index: int):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "20"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([t.strip() for t in line.split(",")])

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": []}
        time.sleep(0.15)
        self.proc.terminate()
        self.thread.join(timeout=2)
        sm = [float(r[0]) for r in self.rows if len(r) >= 6 and r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in self.rows if len(r) >= 6 and r[1].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for i, n in enumerate(names) if any(len(r) >= 6 and r[2 + i].lower().startswith("active") for r in self.rows)]
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": reasons, "samples": len(sm)}


# --------------------------------------------------------------------------------------------------
def cpu_oracle_pass(scale_div: int = 4, quiet=False, openmp=False):
    """One pass of the same hot path by the CPU oracle on a bounded sample (every size / scale_div).
    Returns (algorithmic bytes, seconds, threads, description). openmp: the OpenMP build of the same
    loops; Reduce and Scan stay sequential in it (their order is part of the oracle)."""
    import oracle as O
    import skel_inputs as I
    O.use_openmp(openmp)
    n = (1 << 26) // scale_div
    n28 = (1 << 28) // scale_div
    side = int(8192 / np.sqrt(scale_div))
    x, y = I.uniform_pm1_f32(1, n), I.uniform_pm1_f32(2, n)
    vi = I.uniform_int_i32(3, n, 1000)
    s = I.uniform01_f32(4, n)
    X = I.uniform01_f32(5, side * side).reshape(side, side)
    sc = I.uniform_int_i32(6, n28, 15)
    w = {r: I.positive_weights_f32(10 + r, 2 * r + 1) for r in (1, 4, 8, 16)}
    W5, W9 = I.positive_weights_f32(20, 25), I.positive_weights_f32(21, 81)
    t0 = time.perf_counter()
    nbytes = 0
    O.map_f32(O.FN_SAXPY, 2.5, x, y); nbytes += 12 * n
    O.reduce_i32(O.FN_ADD, vi); O.reduce_i32(O.FN_MAX, vi); nbytes += 8 * n
    O.mapreduce_f32(O.FN_MULT, O.FN_ADD, 0.0, x, y); nbytes += 8 * n
    for r in (1, 4, 16):
        for edge in (O.EDGE_CONSTANT, O.EDGE_DUPLICATE):
            O.mapoverlap_1d(w[r], r, edge, 0.0, s); nbytes += 8 * n
    O.mapoverlap_2d(W5, 2, 2, O.EDGE_DUPLICATE, 0.0, X); nbytes += 8 * side * side
    O.mapoverlap_2d(W9, 4, 4, O.EDGE_DUPLICATE, 0.0, X); nbytes += 8 * side * side
    T, _ = O.mapoverlap_1d_matrix(w[8], 8, O.EDGE_DUPLICATE, 0.0, O.AXIS_ROW, X); nbytes += 8 * side * side
    O.mapoverlap_1d_matrix(w[8], 8, O.EDGE_DUPLICATE, 0.0, O.AXIS_COL, T); nbytes += 8 * side * side
    O.scan_i32(O.FN_ADD, O.SCAN_INCLUSIVE, 0, sc); O.scan_i32(O.FN_ADD, O.SCAN_EXCLUSIVE, 0, sc); nbytes += 16 * n28
    dt = time.perf_counter() - t0
    build = "OpenMP build (-fopenmp)" if openmp else "single-thread build"
    desc = (f"one pass of all skeletons, each at 1/{scale_div} of its bench size (vectors 2^26/{scale_div}, scan "
            f"2^28/{scale_div}, matrix {side}^2), {build} of oracle/oracle.cpp as it stands")
    threads = O.threads()
    O.use_openmp(False)
    return nbytes, dt, threads, desc


def pipeline_experiment(S, ctx, n, iters=100, eager_iters=10):
    """BASELINE.json configs[4], second half: 100 chained calls Map(x*1.0001) -> MapOverlap1D(r=4) ->
    Reduce(sum) on one fp32 smart_vector of n elements (reading 15). Reports what the
    smart containers save: transfers and wall time with the coherence protocol (LAZY) against the
    "no smart containers" baseline (EAGER, run for fewer iterations; per-iteration figures)."""
    import torch
    import skel_inputs as I
    x0 = I.uniform01_f32(I.config_seed(5, 1), n)
    w = I.positive_weights_f32(I.config_seed(3, 14), 9)

    def run(k, lag=0):
        """lag = 0: blocking skel_reduce every iteration. lag > 0: skel_reduce_async, the scalar of iteration i is
        waited for at iteration i + lag (skel_future_wait: an event behind THAT kernel), so `lag` iterations stay in
        flight and the host never drains the stream."""
        a, b = ctx.vector_from(x0), ctx.vector(n)
        ctx.reset_stats()
        e0, e1, es = (torch.cuda.Event(enable_timing=True) for _ in range(3))
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        e0.record()
        s = 0.0
        futs = []
        for it in range(k):
            if it == 1:
                es.record()  # iteration 1 carried the one upload of A (256 MiB over PCIe): steady state starts here
            ctx.map(S.FN_MULT, 1.0001, a, None, a)
            ctx.mapoverlap_1d(w, 4, S.EDGE_DUPLICATE, 0.0, a, b)
            if lag:
                futs.append(ctx.reduce_async(S.FN_ADD, b))
                if len(futs) > lag:
                    s = futs.pop(0).result()
            else:
                s = ctx.reduce(S.FN_ADD, b)
            a, b = b, a
        for f in futs:
            s = f.result()
        e1.record()
        torch.cuda.synchronize()
        wall = time.perf_counter() - t0
        st = ctx.stats()
        a.destroy()
        b.destroy()
        run.steady_ms = es.elapsed_time(e1) / (k - 1) if k > 1 else float("nan")
        return wall, e0.elapsed_time(e1), st, s

    run(3)  # warm-up (allocations, first-use kernel loads)
    wall_l, dev_l, st_l, s_l = run(iters)
    steady_l = run.steady_ms
    # the same loop with cross-call fusion on (skel_ctx_set_fusion): Map -> MapOverlap1D -> Reduce is ONE
    # kernel, 12 instead of 20 bytes per element (every reduce() ends with a scalar read-back, which also
    # flushes: the events above see every launch)
    wall_la, dev_la, st_la, s_la = run(iters, lag=2)
    steady_la = run.steady_ms
    ctx.set_fusion(True)
    try:
        run(3)
        wall_f, dev_f, st_f, s_f = run(iters)
        steady_f = run.steady_ms
        run(3, lag=2)
        wall_fa, dev_fa, st_fa, s_fa = run(iters, lag=2)
        steady_fa = run.steady_ms
    finally:
        ctx.set_fusion(False)
    ctx.set_coherence(S.EAGER)
    try:
        wall_e, _, st_e, _ = run(eager_iters)
    finally:
        ctx.set_coherence(S.LAZY)
    per_iter_bytes = 20 * n  # Map 8 + MapOverlap 8 + Reduce 4 bytes per element
    return {
        "n": n, "iterations": iters,
        "note": "wall / device per iteration include the ONE upload of A (256 MiB over PCIe, ~5 ms) spread over the "
                "iterations; steady_device_ms_per_iter is iterations 2..100 only",
        "lazy": {"wall_ms_per_iter": round(wall_l / iters * 1e3, 4), "device_ms_per_iter": round(dev_l / iters, 4),
                 "steady_device_ms_per_iter": round(steady_l, 4),
                 "GB/s_device": round(per_iter_bytes / (dev_l / iters * 1e-3) / 1e9, 1),
                 "h2d_bytes_total": st_l["h2d_bytes"], "d2h_bytes_total": st_l["d2h_bytes"],
                 "h2d_count": st_l["h2d_count"], "d2h_count": st_l["d2h_count"],
                 "scalar_readbacks": st_l["scalar_d2h_count"], "h2d_elided": st_l["h2d_elided"]},
        "lazy_async": {"wall_ms_per_iter": round(wall_la / iters * 1e3, 4), "device_ms_per_iter": round(dev_la / iters, 4),
                       "steady_device_ms_per_iter": round(steady_la, 4),
                       "iterations_in_flight": 2, "scalar_readbacks": st_la["scalar_d2h_count"],
                       "same_scalar_as_blocking": bool(s_la == s_l),
                       "note": "skel_reduce_async + skel_future_wait two iterations late: the host waits on the event "
                               "behind each reducing kernel, never on the whole stream"},
        "fused": {"wall_ms_per_iter": round(wall_f / iters * 1e3, 4), "device_ms_per_iter": round(dev_f / iters, 4),
                  "steady_device_ms_per_iter": round(steady_f, 4),
                  "bytes_per_elem": 12, "GB/s_device_at_12B": round(12 * n / (dev_f / iters * 1e-3) / 1e9, 1),
                  "launches_per_iter": st_f["launches"] / iters, "fused_launches": st_f["fused_launches"],
                  "h2d_count": st_f["h2d_count"], "d2h_count": st_f["d2h_count"],
                  "speedup_over_unfused_device": round(dev_l / dev_f, 3), "last_scalar": s_f},
        "fused_async": {"wall_ms_per_iter": round(wall_fa / iters * 1e3, 4), "device_ms_per_iter": round(dev_fa / iters, 4),
                        "steady_device_ms_per_iter": round(steady_fa, 4),
                        "steady_GB/s_at_12B": round(12 * n / (steady_fa * 1e-3) / 1e9, 1),
                        "iterations_in_flight": 2, "launches_per_iter": st_fa["launches"] / iters,
                        "scalar_readbacks": st_fa["scalar_d2h_count"], "same_scalar_as_blocking": bool(s_fa == s_f),
                        "GB/s_wall_at_12B": round(12 * n / (wall_fa / iters) / 1e9, 1)},
        "eager": {"iterations_run": eager_iters, "wall_ms_per_iter": round(wall_e / eager_iters * 1e3, 3),
                  "h2d_bytes_per_iter": st_e["h2d_bytes"] // eager_iters, "d2h_bytes_per_iter": st_e["d2h_bytes"] // eager_iters,
                  "transfers_per_iter": (st_e["h2d_count"] + st_e["d2h_count"]) // eager_iters},
        "speedup_lazy_over_eager": round((wall_e / eager_iters) / (wall_l / iters), 1),
        "closed_form": {"lazy_h2d_bytes": 4 * n, "lazy_d2h_bytes": 0, "eager_bytes_per_iter": 5 * 4 * n},
        "last_scalar": s_l,
    }


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle as O
    O.build()
    times = []
    nbytes = desc = None
    for i in range(args.warmup + args.steps):
        nbytes, dt, threads, desc = cpu_oracle_pass(args.ref_div)
        if i >= args.warmup:
            times.append(dt)
    t = float(np.mean(times))
    v = nbytes / t / 1e9
    line = {"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": t * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic (seeded, BASELINE.json configs)",
            "config": {"workload": "all skeletons at BASELINE.json configs[1..4] sizes, bounded sample for the CPU oracle"},
            "cpu_baseline": {"value": v, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": desc},
            "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# --------------------------------------------------------------------------------------------------
def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=30)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours")
    ap.add_argument("--scale", type=float, default=1.0, help="shrink every size (testing only; <1 invalidates the number)")
    ap.add_argument("--ref-div", type=int, default=8)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-pipeline", action="store_true")
    ap.add_argument("--force", action="append", default=[], metavar="SKELETON_ID=VARIANT_ID",
                    help="force a kernel variant for a skeleton id (profiling aid), e.g. --force 3=3")
    ap.add_argument("--plan", default=os.path.join(ROOT, "paper_1405_2915_b200", "plans", "b200.plan"))
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl != "reference" else args.warmup
    if args.impl == "reference":
        return run_reference(args)

    import torch
    from paper_1405_2915_b200.replicas import Replicas, env_world
    world, rank, local = env_world()
    torch.cuda.set_device(local)
    rep = Replicas("nccl", torch.device("cuda", local))  # replicas only: barrier + max-over-ranks timing
    from paper_1405_2915_b200 import skel as S  # fails loudly if libskel.so is missing

    sz = sizes(args.scale)
    d = gen_inputs(sz)
    ctx = S.Context()
    if args.plan and os.path.exists(args.plan):
        ctx.plan_load(args.plan)
    for f in args.force:
        sk, v = f.split("=")
        ctx.force_variant(int(sk), int(v))
    wl = Workload(S, ctx, d, sz)
    nops = len(wl.ops)

    def barrier():
        torch.cuda.synchronize()
        rep.barrier()
        torch.cuda.synchronize()

    # ---- device-resident timing
    for _ in range(args.warmup):
        wl.step()
    barrier()
    ev = [[(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(nops)]
          for _ in range(args.steps)]
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    sampler = ClockSampler(local)
    sampler.start()
    # untimed pre-roll of the same steps while nvidia-smi starts up (its first sample takes ~0.2 s), so that
    # the clock / throttle samples are taken under the load of the timed region, not on an idle GPU
    t_pre = time.perf_counter()
    while time.perf_counter() - t_pre < 0.5:
        wl.step()
        torch.cuda.synchronize()
    ctx.reset_stats()
    barrier()
    e0.record()
    for k in range(args.steps):
        wl.step(ev[k])
    e1.record()
    barrier()
    clocks = sampler.stop()
    launches = ctx.stats()["launches"]
    value, ms_per_step = rep.aggregate_throughput(wl.bytes_per_step, e0.elapsed_time(e1) / args.steps)
    value /= 1e9
    wl.verify(d)

    # per-call breakdown (median over steps)
    peak, peak_src = measured_peaks()
    per = {}
    kern_time = {}  # kernel (one template instantiation; edge policy / scan mode are run-time arguments) -> totals

    def kernel_key(name):
        for suffix in ("_const0", "_dup", "_inclusive_i32", "_exclusive_i32"):
            if name.endswith(suffix):
                return name[: -len(suffix)]
        return name

    for i, (name, fam, _, nbytes, elems) in enumerate(wl.ops):
        ts = sorted(ev[k][i][0].elapsed_time(ev[k][i][1]) for k in range(args.steps))
        med = ts[len(ts) // 2]
        mean = float(np.mean(ts))
        # us = median; us_mean = mean over the steps: CUDA event timestamps tick in steps of about 2 us on this driver,
        # so the median of 30 samples is quantised to that step and the mean is the finer figure
        per[name] = {"us": round(med * 1e3, 2), "us_mean": round(mean * 1e3, 2), "GB/s": round(nbytes / (med * 1e-3) / 1e9, 1),
                     "Gelem/s": round(elems / (med * 1e-3) / 1e9, 1), "frac_measured_hbm": round(nbytes / (med * 1e-3) / 1e9 / peak, 4),
                     "frac_8TBs": round(nbytes / (med * 1e-3) / 1e9 / 8000.0, 4), "variant": None}
        kt = kern_time.setdefault(kernel_key(name), [0.0, 0, 0])
        kt[0] += mean
        kt[1] += nbytes
        kt[2] += 1
    # variant names actually chosen
    for i, (name, fam, fn, _, _) in enumerate(wl.ops):
        fn()
        sk, v = ctx.last_variant()
        per[name]["variant"] = S.variant_names(sk)[v]
    ctx.sync()
    dom = max(kern_time, key=lambda f: kern_time[f][0])
    dt_ms, dbytes, dcount = kern_time[dom]
    achieved = dbytes / (dt_ms * 1e-3) / 1e9
    dom_ops = [name for name, *_ in wl.ops if kernel_key(name) == dom]
    dom_variant = per[dom_ops[0]]["variant"]
    roofline = {"bound": "hbm", "kernel": dom, "variant": dom_variant, "achieved": round(achieved, 1), "peak": peak, "unit": "GB/s",
                "frac": round(achieved / peak, 4),
                "traffic": ncu_traffic(dom_ops[0], dom_variant) if args.scale == 1.0 else None,
                "traffic_source": "profiles/r02_ncu_traffic.csv (ncu --set full, per launch, keyed by variant)",
                "algorithmic_bytes_per_launch": dbytes // dcount,
                "peak_source": peak_src, "launches_per_step": dcount, "avg_launch_us": round(dt_ms * 1e3 / dcount, 2),
                "share_of_step": round(dt_ms / ms_per_step, 4)}

    # ---- arithmetic roofline of the MapOverlap rows: FMAs per element over the FP32 FMA rate
    # measured in this run by a register-only FFMA kernel; "bound" = the larger of the two floors
    fma_peak = ctx.probe_fma_peak(5)  # FMA/s
    # what a shared-memory load costs the FMA pipe: FFMA2 stream + NL LDS.128 per 144 pipe cycles
    fma_vs_loads = {f"lds128_per_144_cycles={nl}": round(ctx.probe_fma_with_loads(nl, 5) / 1e12, 2) for nl in (0, 1, 2, 4, 8)}
    fma_per_elem = {"overlap1d_r1": 3, "overlap1d_r4": 9, "overlap1d_r16": 33, "overlap2d_5x5": 25, "overlap2d_9x9": 81,
                    "overlap1d_rows_r8": 17, "overlap1d_cols_r8": 17}
    for name, _, _, nbytes, elems in wl.ops:
        for key, f in fma_per_elem.items():
            if name.startswith(key):
                alu_us = elems * f / fma_peak * 1e6
                hbm_us = nbytes / (peak * 1e9) * 1e6
                per[name].update({"fma_per_elem": f, "alu_floor_us": round(alu_us, 1), "hbm_floor_us": round(hbm_us, 1),
                                  "bound": "alu" if alu_us > hbm_us else "hbm",
                                  "frac_fma_roofline": round(alu_us / per[name]["us"], 4)})

    # ---- small-n latency (config 0: dot n = 2^20, L2 resident) — reported, not part of `value`
    import skel_inputs as I
    n20 = 1 << 20
    a20, b20 = ctx.vector_from(I.uniform_pm1_f32(I.config_seed(1, 0), n20)), ctx.vector_from(I.uniform_pm1_f32(I.config_seed(1, 1), n20))
    for _ in range(5):
        ctx.mapreduce_to(S.FN_MULT, S.FN_ADD, 0.0, a20, b20, wl.resf, 1)
    s0, s1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    s0.record()
    for _ in range(50):
        ctx.mapreduce_to(S.FN_MULT, S.FN_ADD, 0.0, a20, b20, wl.resf, 1)
    s1.record()
    torch.cuda.synchronize()
    dot20_us = s0.elapsed_time(s1) * 1e3 / 50
    a20.destroy()
    b20.destroy()

    # ---- chained pipeline / transfer elision (reported, not part of `value`)
    pipeline = None
    if rank == 0 and not args.no_pipeline:
        pipeline = pipeline_experiment(S, ctx, sz["n26"])

    # ---- fused separable MapOverlap (reported, not part of `value`: the step keeps the two 1D calls of
    # BASELINE.json configs[3]); same matrix, same filters, one call instead of two
    separable = None
    if rank == 0 and not args.no_pipeline:
        import torch
        m = sz["side"] * sz["side"]
        call = lambda: ctx.mapoverlap_separable(d["wr8"], 8, d["wc8"], 8, S.EDGE_DUPLICATE, 0.0, wl.mX, wl.mO)  # noqa: E731
        for _ in range(3):
            call()
        ts = []
        for _ in range(20):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            call()
            e1.record()
            e1.synchronize()
            ts.append(e0.elapsed_time(e1) * 1e3)
        us = float(np.median(ts))
        two = per["overlap1d_rows_r8_dup"]["us"] + per["overlap1d_cols_r8_dup"]["us"]
        separable = {"us": round(us, 2), "variant": S.variant_names(S.SK_SEPARABLE)[ctx.last_variant()[1]],
                     "bytes_per_elem": 8, "GB/s_at_8B": round(8 * m / us / 1e3, 1),
                     "frac_measured_hbm": round(8 * m / us / 1e3 / peak, 4),
                     "two_calls_us": round(two, 2), "speedup_over_two_calls": round(two / us, 3)}
        # the same pair with CONSTANT 0 edges: the register-marching form (csrc/separable.cu "march_r8") needs no border pass there
        callc = lambda: ctx.mapoverlap_separable(d["wr8"], 8, d["wc8"], 8, S.EDGE_CONSTANT, 0.0, wl.mX, wl.mO)  # noqa: E731
        for _ in range(3):
            callc()
        ts = []
        for _ in range(20):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            callc()
            e1.record()
            e1.synchronize()
            ts.append(e0.elapsed_time(e1) * 1e3)
        usc = float(np.median(ts))
        separable["const0_edges"] = {"us": round(usc, 2), "variant": S.variant_names(S.SK_SEPARABLE)[ctx.last_variant()[1]],
                                     "GB/s_at_8B": round(8 * m / usc / 1e3, 1), "frac_measured_hbm": round(8 * m / usc / 1e3 / peak, 4)}

    # ---- row-wise Reduce on the 8192^2 matrix (reported, not part of `value`)
    reduce_rows = map3 = None
    if rank == 0 and not args.no_pipeline:
        import torch
        m = sz["side"] * sz["side"]
        rr = ctx.vector(sz["side"])
        call = lambda: ctx.reduce_rows(S.FN_ADD, wl.mX, rr)  # noqa: E731
        for _ in range(3):
            call()
        ts = []
        for _ in range(20):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            call()
            e1.record()
            e1.synchronize()
            ts.append(e0.elapsed_time(e1) * 1e3)
        us = float(np.median(ts))
        rows_variant = S.variant_names(S.SK_REDUCE_ROWS)[ctx.last_variant()[1]]
        got = rr.numpy()
        ref = d["X"].astype(np.float64).sum(axis=1)
        assert np.all(np.abs(got - ref) <= 1e-5 * np.abs(d["X"]).astype(np.float64).sum(axis=1)), "reduce_rows mismatch"
        # three-vector Map (MULADD) on the step's vectors: 16 B/elem
        n26 = sz["n26"]
        call3 = lambda: ctx.map3(S.FN_MULADD, wl.vx, wl.vy, wl.vs, wl.vr)  # noqa: E731
        for _ in range(3):
            call3()
        t3 = []
        for _ in range(20):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            call3()
            e1.record()
            e1.synchronize()
            t3.append(e0.elapsed_time(e1) * 1e3)
        us3 = float(np.median(t3))
        map3 = {"us": round(us3, 2), "variant": S.variant_names(S.SK_MAP)[ctx.last_variant()[1]], "bytes_per_elem": 16,
                "GB/s": round(16 * n26 / us3 / 1e3, 1), "frac_measured_hbm": round(16 * n26 / us3 / 1e3 / peak, 4)}
        reduce_rows = {"us": round(us, 2), "variant": rows_variant,
                       "bytes_per_elem": 4, "GB/s": round(4 * m / us / 1e3, 1), "frac_measured_hbm": round(4 * m / us / 1e3 / peak, 4)}
        rr.destroy()

    # ---- the other element types: int32 MapOverlap and fp64 skeletons at the bench sizes. Not part
    # of `value` (BASELINE.json's configs are f32 / i32 Reduce / i32 Scan); same timing protocol, each call preceded
    # by nothing but its own previous launch (working sets > L2).
    other_dtypes = None
    if rank == 0 and not args.no_pipeline:
        import torch
        import skel_inputs as I

        def timed(call, reps=15):
            for _ in range(3):
                call()
            ts = []
            for _ in range(reps):
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record()
                call()
                e1.record()
                e1.synchronize()
                ts.append(e0.elapsed_time(e1) * 1e3)
            return float(np.median(ts))

        def row(us, nbytes, sk, f64=False):
            return {"us": round(us, 2), "GB/s": round(nbytes / us / 1e3, 1), "frac_measured_hbm": round(nbytes / us / 1e3 / peak, 4),
                    "variant": "f64 (one kernel per skeleton, csrc/f64.cu)" if f64 else S.variant_names(sk)[ctx.last_variant()[1]]}

        other_dtypes = {}
        n26, side = sz["n26"], sz["side"]
        vi_o = ctx.vector(n26, S.I32)
        wi4 = (I.uniform_int_i32(31, 9, 200) - 100).astype(np.int32)
        us = timed(lambda: ctx.mapoverlap_1d_i32(wi4, 4, S.EDGE_DUPLICATE, 0, wl.vi, vi_o))
        other_dtypes["overlap1d_r4_dup_i32"] = row(us, 8 * n26, S.SK_OVERLAP1D)
        vi_o.destroy()
        Xi = I.uniform_int_i32(32, side * side, 1000).reshape(side, side)
        mi, mio = ctx.matrix_from(Xi), ctx.matrix(side, side, S.I32)
        Wi = (I.uniform_int_i32(33, 25, 200) - 100).astype(np.int32)
        us = timed(lambda: ctx.mapoverlap_2d_i32(Wi, 2, 2, S.EDGE_DUPLICATE, 0, mi, mio))
        other_dtypes["overlap2d_5x5_dup_i32"] = row(us, 8 * side * side, S.SK_OVERLAP2D)
        mi.destroy()
        mio.destroy()
        n25 = n26 // 2   # the same bytes per operand as the f32 vectors
        xd, yd = ctx.vector_from(I.uniform_pm1_f64(34, n25)), ctx.vector_from(I.uniform_pm1_f64(35, n25))
        od, rd = ctx.vector(n25, S.F64), ctx.vector(2, S.F64)
        us = timed(lambda: ctx.map(S.FN_SAXPY, 2.5, xd, yd, od))
        other_dtypes["map_saxpy_f64"] = row(us, 24 * n25, S.SK_MAP, True)
        us = timed(lambda: ctx.mapreduce_to(S.FN_MULT, S.FN_ADD, 0.0, xd, yd, rd, 0))
        other_dtypes["mapreduce_dot_f64"] = row(us, 16 * n25, S.SK_MAPREDUCE, True)
        us = timed(lambda: ctx.scan(S.FN_ADD, S.SCAN_INCLUSIVE, 0.0, xd, od))
        other_dtypes["scan_inclusive_f64"] = dict(row(us, 16 * n25, S.SK_SCAN, True), note="single pass over HBM (l2ahead form, f64.cu), the tile is re-read from L2")
        wd = I.uniform_pm1_f64(36, 9)
        us = timed(lambda: ctx.mapoverlap_1d_f64(wd, 4, S.EDGE_DUPLICATE, 0.0, xd, od))
        other_dtypes["overlap1d_r4_dup_f64"] = dict(row(us, 16 * n25, S.SK_OVERLAP1D, True), note="256-bit row form (f64.cu)")
        for c in (xd, yd, od, rd):
            c.destroy()

    # ---- range-granular host access (PAPER.md L123 partial copies): the host updates 1 MiB of a
    # 256 MiB vector between two Reduce calls; with a range access only that MiB is uploaded, with the whole-container
    # protocol (READWRITE access to the container) the device copy is invalidated and 256 MiB go up again
    range_update = None
    if rank == 0 and not args.no_pipeline:
        nr = 1 << 18
        patch = np.full(nr, 0.5, np.float32)

        def upd(ranged):
            ctx.reset_stats()
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            for it in range(5):
                if ranged:
                    wl.vs.write_range(4096 * (it + 1), patch)
                else:
                    hv = wl.vs.host_view(S.READWRITE)
                    hv[4096 * (it + 1):4096 * (it + 1) + nr] = patch
                    wl.vs.release()
                ctx.reduce(S.FN_ADD, wl.vs)
            dt = (time.perf_counter() - t0) / 5
            return dt, ctx.stats()

        ctx.reduce(S.FN_ADD, wl.vs)
        wl.vs.numpy()  # host copy valid too (SHARED): both protocols start from the same state
        upd(True)
        t_r, st_r = upd(True)
        t_w, st_w = upd(False)
        range_update = {"range_bytes": 4 * nr, "container_bytes": 4 * sz["n26"],
                        "range_access": {"ms_per_update_and_reduce": round(t_r * 1e3, 3), "h2d_bytes_per_update": st_r["h2d_bytes"] // 5},
                        "whole_container_access": {"ms_per_update_and_reduce": round(t_w * 1e3, 3), "h2d_bytes_per_update": st_w["h2d_bytes"] // 5},
                        "speedup": round(t_w / t_r, 1)}

    # ---- container-layer overhead ("< 1 %") and the dot-product size sweep
    # (SURVEY.md 8(d) cfg 1): reported, not part of `value`
    container_layer = dot_sweep = None
    if rank == 0 and not args.no_pipeline:
        import torch
        enq = []
        for _ in range(10):  # host time to ENQUEUE one step (16 asynchronous calls), device idle at the start
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            wl.step()
            enq.append(time.perf_counter() - t0)
            torch.cuda.synchronize()
        host_ms = float(np.median(enq)) * 1e3
        # SURVEY.md 8(d)(4) / PAPER.md L123 ("negligible (less than 1 %)"): the SAME 16 kernel launches through the
        # container layer against bare launches on raw device pointers, both timed inside the library (no Python, no
        # ctypes): skel_replay_* records the step's calls and replays them either way.
        ctx.replay_begin()
        wl.step()
        ncalls = ctx.replay_end()
        for raw in (False, True):
            ctx.replay_run(raw, 3)
        hc, dc, hr, dr = [], [], [], []
        for _ in range(5):  # interleaved: clock / power drift hits both alike
            h, dv = ctx.replay_run(False, 10)
            hc.append(h), dc.append(dv)
            h, dv = ctx.replay_run(True, 10)
            hr.append(h), dr.append(dv)
        hc, dc, hr, dr = (float(np.median(v)) for v in (hc, dc, hr, dr))
        container_layer = {
            "definition": "time of one step (16 calls) through skel_* on containers / time of the same 16 kernel "
                          "launches on raw device pointers - 1 (SURVEY.md 8(d)(4)); timed in C inside libskel.so",
            "calls": ncalls,
            "device_us_per_step_containers": round(dc, 2), "device_us_per_step_raw": round(dr, 2),
            "device_overhead": round(dc / dr - 1.0, 5),
            "host_us_per_step_containers": round(hc, 2), "host_us_per_step_raw": round(hr, 2),
            "host_us_per_call_containers": round(hc / ncalls, 3), "host_us_per_call_raw": round(hr / ncalls, 3),
            "host_overhead_us_per_call": round((hc - hr) / ncalls, 3),
            "host_enqueue_fraction_of_device_time": round(hc / dc, 5),
            "paper_claim": "< 1 % (PAPER.md L123)",
            "through_python_ctypes": {"host_us_per_call": round(host_ms * 1e3 / nops, 2), "host_ms_per_step": round(host_ms, 4),
                                      "note": "the same step enqueued from Python: ctypes marshalling included"}}
        nmax = 1 << 28
        tx, ty = torch.rand(nmax, device="cuda") * 2 - 1, torch.rand(nmax, device="cuda") * 2 - 1
        res = ctx.vector(1)
        dot_sweep = {}
        for lg in range(20, 29, 2):
            n = 1 << lg
            va, vb = ctx.vector_adopt(tx[:n]), ctx.vector_adopt(ty[:n])
            call = lambda: ctx.mapreduce_to(S.FN_MULT, S.FN_ADD, 0.0, va, vb, res, 0)  # noqa: E731
            for _ in range(3):
                call()
            ts = []
            for _ in range(15):
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record()
                call()
                e1.record()
                e1.synchronize()
                ts.append(e0.elapsed_time(e1) * 1e3)
            us = float(np.median(ts))
            dot_sweep[f"2^{lg}"] = {"us": round(us, 2), "GB/s": round(8 * n / us / 1e3, 1),
                                    "frac_measured_hbm": round(8 * n / us / 1e3 / peak, 4),
                                    "l2_resident": 8 * n <= 126 * (1 << 20)}
            va.destroy()
            vb.destroy()
        res.destroy()
        del tx, ty

    # ---- end to end through host buffers
    e2e = None
    if not args.no_e2e:
        wl.e2e_step()
        barrier()
        ctx.reset_stats()
        t0 = time.perf_counter()
        for _ in range(args.steps):
            wl.e2e_step()
        barrier()
        dt = time.perf_counter() - t0
        dt = rep.max_over_ranks(dt)
        st = ctx.stats()
        e2e = {"value": round(world * wl.bytes_per_step * args.steps / dt / 1e9, 2), "unit": UNIT,
               "h2d_bytes_per_step": st["h2d_bytes"] // args.steps, "d2h_bytes_per_step": st["d2h_bytes"] // args.steps,
               "ms_per_step": round(dt / args.steps * 1e3, 2),
               "note": "outputs are prefetched to the host on a copy stream as soon as they are final (skel_*_prefetch_host)"}
        # the same without the prefetch hints (pure lazy protocol: every download starts at the host access)
        wl.e2e_step(prefetch=False)
        barrier()
        t0 = time.perf_counter()
        for _ in range(max(1, args.steps // 3)):
            wl.e2e_step(prefetch=False)
        barrier()
        dt2 = rep.max_over_ranks(time.perf_counter() - t0) / max(1, args.steps // 3)
        e2e["without_prefetch"] = {"value": round(world * wl.bytes_per_step / dt2 / 1e9, 2), "ms_per_step": round(dt2 * 1e3, 2)}

    cpu = cpu_omp = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        nb, dt, threads, desc = cpu_oracle_pass(2)
        cpu = {"value": round(nb / dt / 1e9, 3), "unit": UNIT, "cores": threads, "kind": "oracle", "sample": desc,
               "seconds": round(dt, 2), "host_cores_available": os.cpu_count()}
        nb, dt, threads, desc = cpu_oracle_pass(2, openmp=True)
        cpu_omp = {"value": round(nb / dt / 1e9, 3), "unit": UNIT, "cores": threads, "kind": "oracle", "sample": desc,
                   "seconds": round(dt, 2)}

    if rank == 0:
        line = {"metric": METRIC, "value": round(value, 1), "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": args.warmup, "ms_per_step": round(ms_per_step, 4), "higher_is_better": True, "scaling": "weak",
                "vs_baseline": None, "dtype": "f32+i32", "data": "synthetic (seeded counter-based generator, BASELINE.json configs)",
                "config": {"workload": "all skeletons at their largest BASELINE.json config (configs[1..4]): Map saxpy 2^26, "
                                       "Reduce sum+max i32 2^26, MapReduce dot 2^26, MapOverlap1D r{1,4,16}x{const0,dup} 2^26, "
                                       "MapOverlap2D 5x5/9x9 + separable r8 on 8192^2, Scan incl+excl i32 2^28",
                           "scale": args.scale, "l2": "every working set > 126 MB L2; no flush", "calls_per_step": nops,
                           "bytes_per_step": wl.bytes_per_step, "parallelism": "replicas only" if world > 1 else "1 GPU"},
                "Gelem/s": round(world * wl.elems_per_step / (ms_per_step * 1e-3) / 1e9, 1),
                "frac_measured_hbm": round(value / world / peak, 4), "frac_8TBs": round(value / world / 8000.0, 4),
                "roofline": roofline, "cpu_baseline": cpu, "e2e": e2e, "gpu_launches": launches, "clocks": clocks,
                "dot_2p20_us_l2_resident": round(dot20_us, 2), "pipeline": pipeline, "separable_fused": separable, "reduce_rows": reduce_rows, "map3_muladd": map3, "other_element_types": other_dtypes, "range_update": range_update,
                "fma_peak_tfma_s": round(fma_peak / 1e12, 2), "fma_tfma_s_vs_shared_loads": fma_vs_loads, "container_layer": container_layer, "dot_sweep": dot_sweep, "cpu_baseline_omp": cpu_omp,
                "per_skeleton": per}
        print(json.dumps(line), flush=True)
    wl.destroy()
    ctx.close()
    rep.close()


if __name__ == "__main__":
    main()
