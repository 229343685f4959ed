#!/usr/bin/env python
"""bench.py — throughput of the Voronoi topological-change hot path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload cfg5]

One "step" = one frame through the whole site-driven hot path:
vor_build_cells -> vor_label -> vor_edges -> vor_diff against the previous frame.  The workload is
BASELINE.json config 5 (16384^2 lattice, 10^6 sites, the configuration the metric is quoted on).
Prints ONE JSON line (rank 0).  See DESIGN.md §8 for the definition of every field.
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

from paper_1607_00908_b200 import workloads as W  # noqa: E402

METRIC = "lattice cells/s labelled+edge-extracted+diffed (frames/s = value / L^2)"
UNIT = "cells/s"


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="cfg5", help="cfg5 (default) | cfg2 | cfg5@L e.g. cfg5@4096")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--cpu-sample-L", type=int, default=0,
                    help="lattice side of the oracle's sample (0 = full workload for ours, 4096 for reference)")
    return ap.parse_args()


def get_workload(name: str):
    if "@" in name:
        base, L = name.split("@")
        return W.scaled(int(base[3:]), int(L))
    return W.config(int(name[3:]))


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json)", float(d.get("sm_max_mhz", 1965.0))
    return 6650.0, "fallback (B200_PROFILING.md)", 1965.0


class ClockSampler:
    """Samples nvidia-smi SM clocks and throttle reasons DURING the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                 "-lms", "100"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append(line.strip())

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            f = [t.strip() for t in r.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1]))
            except ValueError:
                continue
            for n, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


# ------------------------------------------------------------------------------------------ oracle legs
def oracle_frame_seconds(w, frames):
    """Time the oracle, as it stands, on `frames` (list of (sx, sy)); returns (seconds, cells)."""
    import oracle
    prev = np.empty(0, np.uint64)
    t0 = time.perf_counter()
    for sx, sy in frames:
        lab = oracle.label_cells(w.L, sx, sy, w.bucket_cells)
        e = oracle.edges(lab)
        oracle.diff(prev, e)
        prev = e
    return time.perf_counter() - t0, len(frames) * w.L * w.L


def run_reference(args, w):
    """--impl reference: the CPU oracle on the box's host cores (rank 0 only)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    Ls = args.cpu_sample_L or min(4096, w.L)
    ws = w if Ls == w.L else W.scaled(5, Ls) if w.kind == "jittered_grid" else w
    frames = list(ws.frames(args.warmup + args.steps))
    for sx, sy in frames[:args.warmup]:
        oracle.edges(oracle.label_cells(ws.L, sx, sy, ws.bucket_cells))
    secs, cells = oracle_frame_seconds(ws, frames[args.warmup:])
    cores = oracle.num_threads()
    val = cells / secs
    sample = (f"{args.steps} frames of {ws.name} ({ws.L}^2 cells, {ws.n_sites} sites: same density and "
              f"structure as {w.name}); label_cells + edges + diff")
    out = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
           "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * secs / args.steps,
           "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "int64",
           "data": "synthetic", "config": {"workload": w.name, "L": w.L, "n_sites": w.n_sites,
                                           "sample_L": ws.L, "sample_sites": ws.n_sites},
           "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
           "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
           "gpu_launches": 0}
    print(json.dumps(out), flush=True)


# ------------------------------------------------------------------------------------------ our arm
def run_ours(args, w):
    import torch
    import torch.distributed as dist
    from paper_1607_00908_b200.binding import Vor

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device (no CPU fallback)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def max_over_ranks(x: float) -> float:
        if world == 1:
            return x
        t = torch.tensor([x], dtype=torch.float64, device="cuda")
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        return float(t.item())

    # weak scaling: every rank processes its own independent frame sequence (no data-path collective)
    import dataclasses
    wr = dataclasses.replace(w, seed=w.seed + 1000 * rank)
    W_, K = args.warmup, args.steps
    frames = list(wr.frames(W_ + K))
    L, n = wr.L, wr.n_sites
    dframes = [(torch.from_numpy(sx).cuda(), torch.from_numpy(sy).cuda()) for sx, sy in frames]

    cap_keys = max(1 << 20, 16 * n)
    v = Vor(L, n, cap_keys)
    cap_e = 4 * n + 1024
    labels = torch.empty(L * L, dtype=torch.int32, device="cuda")
    edges = [torch.empty(cap_e, dtype=torch.int64, device="cuda") for _ in range(2)]
    n_edges = [torch.zeros(1, dtype=torch.int64, device="cuda") for _ in range(2)]
    created = torch.empty(cap_e, dtype=torch.int64, device="cuda")
    destroyed = torch.empty(cap_e, dtype=torch.int64, device="cuda")
    n_c = torch.zeros(1, dtype=torch.int64, device="cuda")
    n_d = torch.zeros(1, dtype=torch.int64, device="cuda")
    stream = torch.cuda.current_stream()
    names = ["build_cells", "label", "edges", "diff"]

    def step(i, ev=None):
        now, prev = i & 1, 1 - (i & 1)
        sx, sy = dframes[i]
        if ev: ev[0].record(stream)
        v.vor_build_cells(sx, sy)
        if ev: ev[1].record(stream)
        v.vor_label(labels)
        if ev: ev[2].record(stream)
        v.vor_edges(labels, edges[now], n_edges[now])
        if ev: ev[3].record(stream)
        v.vor_diff(edges[prev], n_edges[prev], edges[now], n_edges[now], created, destroyed, n_c, n_d)
        if ev: ev[4].record(stream)

    for i in range(W_):
        step(i)
    v.vor_sync_status()
    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(5)] for _ in range(K)]
    t_beg, t_end = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    sampler = ClockSampler(local)
    barrier()
    sampler.start()
    launches0 = v.vor_launch_count()
    t_beg.record(stream)
    for k in range(K):
        step(W_ + k, evs[k])
    t_end.record(stream)
    barrier()
    clocks = sampler.stop()
    launches = v.vor_launch_count() - launches0
    v.vor_sync_status()
    ms_total = max_over_ranks(t_beg.elapsed_time(t_end))
    kernel_ms = {nm: float(np.mean([evs[k][j].elapsed_time(evs[k][j + 1]) for k in range(K)]))
                 for j, nm in enumerate(names)}
    counts = {"n_edges": int(n_edges[(W_ + K - 1) & 1].item()), "n_created": int(n_c.item()),
              "n_destroyed": int(n_d.item())}
    cells_per_step = L * L
    value = world * K * cells_per_step / (ms_total * 1e-3)

    # ---- e2e: the same frames through vor_frame_host (host buffers, H2D + D2H inside the timed region)
    e2e = None
    if not args.no_e2e:
        hc = np.empty(cap_e, np.uint64); hd = np.empty(cap_e, np.uint64); cnt = np.zeros(3, np.int64)
        v.vor_frame_reset()
        for i in range(W_):
            v.vor_frame_host(frames[i][0], frames[i][1], hc, hd, cnt)
        barrier()
        d2h = 0
        t0 = time.perf_counter()
        for k in range(K):
            v.vor_frame_host(frames[W_ + k][0], frames[W_ + k][1], hc, hd, cnt)
            d2h += 8 * (int(cnt[1]) + int(cnt[2])) + 24
        torch.cuda.synchronize()
        secs = max_over_ranks(time.perf_counter() - t0)
        e2e = {"value": world * K * cells_per_step / secs, "unit": UNIT, "ms_per_step": 1e3 * secs / K,
               "h2d_bytes_per_step": 8 * n, "d2h_bytes_per_step": d2h // K,
               "api": "vor_frame_host (C ABI, host buffers; label image stays on the device)"}

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    hbm_peak, peak_src, sm_max_mhz = peaks()
    # dominant kernel = vor_label (one launch per step).  Algorithmic HBM bytes: 4 B/cell written
    # (SURVEY.md §8d); sites are L2-served.  It is ALU/issue-bound, so the HBM fraction is a floor view.
    label_s = kernel_ms["label"] * 1e-3
    label_bytes = 4.0 * cells_per_step
    roofline = {"kernel": "label_tile_kernel", "bound": "hbm", "achieved": label_bytes / label_s / 1e9,
                "peak": hbm_peak, "unit": "GB/s", "frac": label_bytes / label_s / 1e9 / hbm_peak,
                "traffic": None, "peak_source": peak_src,
                "note": "ALU/issue-bound kernel; algorithmic bytes = 4 B/cell label write"}
    edges_bytes = 4.0 * cells_per_step
    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W_,
        "ms_per_step": ms_total / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "int32", "data": "synthetic",
        "config": {"workload": wr.name, "L": L, "n_sites": n, "frames": K,
                   "parallelism": f"{world} independent frame sequences" if world > 1 else "single GPU",
                   "l2_policy": "working set per step (1 GiB label image written then read) exceeds the 126 MB L2"},
        "frames_per_s": world * K / (ms_total * 1e-3),
        "kernel_ms": kernel_ms, "counts": counts,
        "roofline": roofline,
        "rooflines_other": {
            "edges(emit+sort+unique)": {"bound": "hbm", "achieved": edges_bytes / (kernel_ms["edges"] * 1e-3) / 1e9,
                                        "peak": hbm_peak, "unit": "GB/s",
                                        "frac": edges_bytes / (kernel_ms["edges"] * 1e-3) / 1e9 / hbm_peak},
            "diff": {"bound": "hbm", "achieved": 16.0 * counts["n_edges"] / (kernel_ms["diff"] * 1e-3) / 1e9,
                     "peak": hbm_peak, "unit": "GB/s",
                     "frac": 16.0 * counts["n_edges"] / (kernel_ms["diff"] * 1e-3) / 1e9 / hbm_peak}},
        "clocks": clocks, "gpu_launches": int(launches),
    }
    if e2e:
        out["e2e"] = e2e
    if not args.no_cpu_baseline and world == 1:
        import oracle
        Ls = args.cpu_sample_L or w.L
        ws = w if Ls == w.L else W.scaled(5, Ls)
        fr = list(ws.frames(1))
        secs, cells = oracle_frame_seconds(ws, fr)
        out["cpu_baseline"] = {"value": cells / secs, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
                               "sample": f"1 frame of {ws.name} ({ws.L}^2 cells, {ws.n_sites} sites): "
                                         f"label_cells + edges + diff, {secs:.1f} s"}
    print(json.dumps(out), flush=True)
    if world > 1:
        dist.destroy_process_group()


def main():
    args = parse()
    w = get_workload(args.workload)
    if args.impl == "reference":
        run_reference(args, w)
    else:
        run_ours(args, w)


if __name__ == "__main__":
    main()
