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

# Algorithmic integer work of exact labelling per lattice cell: 7 candidate sites (a
# Voronoi region has 6 neighbours on average, plus the owner) x 3 ops (two multiply-adds of the
# distance expansion, one min) + 1 store.
LABEL_OPS_PER_CELL = 22
# dram__bytes_read.sum + dram__bytes_write.sum per launch from the committed `ncu --set full` capture
# (profiles/r1g_full_summary.md); config 5 only.
NCU_TRAFFIC_BYTES = {"label_cta_kernel": 1.035e9, "edges_stream_kernel": 1.098e9, "rows_insert_kernel": 0.082e9,
                     "edges_finish_kernel": 0.094e9, "diff_kernel": 0.048e9}


def edges_bytes(cells, n_edges):
    return 4.0 * cells + 8.0 * n_edges


METRIC = "lattice cells/s labelled+edge-extracted+diffed (frames/s = value / L^2)"
UNIT = "cells/s"


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="cfg5", help="cfg5 (default) | cfg1 | cfg2 | cfg5@L e.g. cfg5@4096 | cfg3 | cfg4 (field path)")
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


# ---- multi-rank host logic (exercised on CPU with gloo by tests/test_bench_ranks.py)
def rank_workload(w, rank: int):
    """Weak scaling: every rank processes its own independent, seeded frame sequence of the same
    configuration (no data-path collective)."""
    import dataclasses
    return dataclasses.replace(w, seed=w.seed + 1000 * rank)


def reduce_max(x: float, world: int, device) -> float:
    """Max over ranks of a per-rank duration (the job is as slow as its slowest rank)."""
    if world == 1:
        return x
    import torch
    import torch.distributed as dist
    t = torch.tensor([x], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(world: int, steps: int, cells_per_step: int, ms_total: float) -> float:
    """Cells all ranks processed / the slowest rank's time."""
    return world * steps * cells_per_step / (ms_total * 1e-3)


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
        return reduce_max(x, world, "cuda")

    wr = rank_workload(w, rank)
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

    # nvidia-smi samples every 100 ms and the K timed steps take ~14 ms: the sampler runs from the
    # warm-up to the end of the e2e leg (the GPU is busy throughout), which contains the timed region
    sampler = ClockSampler(local)
    sampler.start()
    for i in range(W_):
        step(i)
    v.vor_sync_status()
    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(5)] for _ in range(K)]
    t_beg, t_end = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    launches0 = v.vor_launch_count()
    t_beg.record(stream)
    for k in range(K):
        step(W_ + k, evs[k])
    t_end.record(stream)
    barrier()
    launches = v.vor_launch_count() - launches0
    v.vor_sync_status()
    ms_total = max_over_ranks(t_beg.elapsed_time(t_end))
    kernel_ms = {nm: float(np.mean([evs[k][j].elapsed_time(evs[k][j + 1]) for k in range(K)]))
                 for j, nm in enumerate(names)}
    counts = {"n_edges": int(n_edges[(W_ + K - 1) & 1].item()), "n_created": int(n_c.item()),
              "n_destroyed": int(n_d.item())}
    cells_per_step = L * L
    value = whole_job_value(world, K, cells_per_step, ms_total)

    # ---- per-kernel durations: the same K frames again with the library's per-launch CUDA events
    # (recorded on the launching stream); outside the timed region so they cannot perturb `value`
    v.vor_profile_begin()
    for k in range(K):
        step(W_ + k)
    prof = v.vor_profile_end()
    per_kernel = {}
    for nm, ms in prof:
        per_kernel.setdefault(nm, []).append(ms)
    kernel_launch_ms = {nm: float(np.mean(x)) for nm, x in per_kernel.items()}
    kernel_launches_per_step = {nm: len(x) / K for nm, x in per_kernel.items()}

    # ---- event layer (not part of the step): vor_events on the last frame's lists
    i32 = dict(dtype=torch.int32, device="cuda")
    ev_bufs = [torch.empty(n, **i32) for _ in range(4)]
    ev_m, ev_g = torch.zeros(1, **i32), torch.zeros(1, **i32)
    last = (W_ + K - 1) & 1
    def events():
        v.vor_events(edges[1 - last], n_edges[1 - last], edges[last], n_edges[last], created, n_c, destroyed, n_d,
                     ev_bufs[0], ev_bufs[1], ev_m, ev_g, ev_bufs[2], ev_bufs[3])
    for _ in range(3):
        events()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for _ in range(10):
        events()
    e1.record(stream)
    torch.cuda.synchronize()
    events_info = {"ms": e0.elapsed_time(e1) / 10, "events_number": int(ev_m.item()), "global_trigger": int(ev_g.item()),
                   "api": "vor_events: local_trigger, eventsIndices, eventsCount past/now (PAPER.md:215-236)"}

    # ---- e2e: the same frames through vor_frame_host (host buffers, H2D + D2H inside the timed region)
    e2e = None
    if not args.no_e2e:
        # page-locked host buffers (the user's side of the API): inputs are DMA'd straight from them
        def pinned(shape, dtype):
            return torch.empty(shape, dtype=dtype, pin_memory=True).numpy()
        hc = pinned(cap_e, torch.int64).view(np.uint64); hd = pinned(cap_e, torch.int64).view(np.uint64)
        cnt = np.zeros(3, np.int64)
        hframes = []
        for sx, sy in frames:
            px, py = pinned(n, torch.int32), pinned(n, torch.int32)
            px[:] = sx; py[:] = sy
            hframes.append((px, py))
        v.vor_frame_reset()
        for i in range(W_):
            v.vor_frame_host(hframes[i][0], hframes[i][1], hc, hd, cnt)
        barrier()
        t0 = time.perf_counter()
        for k in range(K):
            v.vor_frame_host(hframes[W_ + k][0], hframes[W_ + k][1], hc, hd, cnt)
        torch.cuda.synchronize()
        secs_sync = max_over_ranks(time.perf_counter() - t0)
        # pipelined: frame k+1 is submitted before frame k is collected, so the uploads and downloads
        # (own copy streams) overlap the kernels; every copy is still inside the timed region
        v.vor_frame_reset()
        for i in range(W_):
            v.vor_frame_submit(hframes[i][0], hframes[i][1])
            v.vor_frame_collect(hc, hd, cnt)
        barrier()
        d2h = 0
        t0 = time.perf_counter()
        v.vor_frame_submit(hframes[W_][0], hframes[W_][1])
        for k in range(1, K):
            v.vor_frame_submit(hframes[W_ + k][0], hframes[W_ + k][1])
            v.vor_frame_collect(hc, hd, cnt)
            d2h += 8 * (int(cnt[1]) + int(cnt[2])) + 32
        v.vor_frame_collect(hc, hd, cnt)
        d2h += 8 * (int(cnt[1]) + int(cnt[2])) + 32
        torch.cuda.synchronize()
        secs = max_over_ranks(time.perf_counter() - t0)
        e2e = {"value": world * K * cells_per_step / secs, "unit": UNIT, "ms_per_step": 1e3 * secs / K,
               "h2d_bytes_per_step": 8 * n, "d2h_bytes_per_step": d2h // K,
               "api": "vor_frame_submit / vor_frame_collect (C ABI, pinned host buffers, two frames in flight; "
                      "label image stays on the device)",
               "sync_api_ms_per_step": 1e3 * secs_sync / K,
               "sync_api": "vor_frame_host, one frame at a time (copies not overlapped)"}

    clocks = sampler.stop()
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    hbm_peak, peak_src, sm_max_mhz = peaks()
    # Dominant kernel = label_cta_kernel (one launch per step).  It is bound by plain
    # integer issue, not by HBM: `roofline` reports it against the INT32 lane peak DESIGN.md §5.9
    # derives (SMs x 128 lanes x max SM clock); algorithmic work = 22 integer ops per cell.
    lab_name = max((nm for nm in kernel_launch_ms if "label" in nm), key=lambda nm: kernel_launch_ms[nm])
    label_s = kernel_launch_ms[lab_name] * 1e-3
    alu_peak = 148 * 128 * sm_max_mhz * 1e6 / 1e12            # Tera int32 lane-ops / s
    alu_ops = LABEL_OPS_PER_CELL * cells_per_step
    roofline = {"kernel": lab_name, "bound": "alu", "achieved": alu_ops / label_s / 1e12, "peak": alu_peak,
                "unit": "Tera int32 op/s", "frac": alu_ops / label_s / 1e12 / alu_peak,
                "traffic": NCU_TRAFFIC_BYTES.get(lab_name) if wr.name == "cfg5_throughput_stress" else None,
                "launch_ms": kernel_launch_ms[lab_name],
                "peak_source": "148 SMs x 128 INT32 lanes x max SM clock (DESIGN.md 5.9)",
                "algorithmic": f"{LABEL_OPS_PER_CELL} int32 ops/cell x {cells_per_step} cells",
                "hbm_view": {"achieved": 4.0 * cells_per_step / label_s / 1e9, "peak": hbm_peak, "unit": "GB/s",
                             "frac": 4.0 * cells_per_step / label_s / 1e9 / hbm_peak,
                             "algorithmic": "4 B/cell label write", "peak_source": peak_src}}

    def hbm_roof(name, nbytes, what):
        if name not in kernel_launch_ms:
            return None
        sec = kernel_launch_ms[name] * 1e-3
        return {"bound": "hbm", "achieved": nbytes / sec / 1e9, "peak": hbm_peak, "unit": "GB/s",
                "frac": nbytes / sec / 1e9 / hbm_peak, "launch_ms": kernel_launch_ms[name],
                "traffic": NCU_TRAFFIC_BYTES.get(name) if wr.name == "cfg5_throughput_stress" else None, "algorithmic": what, "peak_source": peak_src}

    ne = counts["n_edges"]
    others = {
        "edges_stream_kernel": hbm_roof("edges_stream_kernel", 4.0 * cells_per_step, "4 B/cell label read"),
        "diff_kernel": hbm_roof("diff_kernel", 16.0 * ne + 8.0 * (counts["n_created"] + counts["n_destroyed"]),
                                "8 B x (E_prev + E_now) read + 8 B x (created + destroyed) written; L2-resident"),
        "vor_edges (stream + insert + finish)": {
            "bound": "hbm", "achieved": edges_bytes(cells_per_step, ne) / (kernel_ms["edges"] * 1e-3) / 1e9,
            "peak": hbm_peak, "unit": "GB/s",
            "frac": edges_bytes(cells_per_step, ne) / (kernel_ms["edges"] * 1e-3) / 1e9 / hbm_peak,
            "algorithmic": "4 B/cell label read + 8 B/edge written"},
    }
    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W_,
        "ms_per_step": ms_total / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "int32", "data": "synthetic",
        "config": {"workload": wr.name, "L": L, "n_sites": n, "frames": K,
                   "parallelism": f"{world} independent frame sequences" if world > 1 else "single GPU",
                   "l2_policy": "working set per step (1 GiB label image written then read) exceeds the 126 MB L2"},
        "frames_per_s": world * K / (ms_total * 1e-3),
        "kernel_ms": kernel_ms, "counts": counts,
        "kernel_launch_ms": kernel_launch_ms, "kernel_launches_per_step": kernel_launches_per_step,
        "roofline": roofline,
        "rooflines_other": {k: r for k, r in others.items() if r},
        "events": events_info,
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


# ------------------------------------------------------------------------------------------ field path
def run_field(args, w):
    """--workload cfg3 | cfg4: one step = one frame of the field-derived path, rows a6..a8 then a1..a5
    (threshold+CCL -> centroids -> match -> cell list -> label -> edges -> diff with maps).  Single GPU;
    not the default bench line (the metric is quoted on config 5) - reported for the §8(a) field rows."""
    import torch
    from paper_1607_00908_b200.binding import Vor
    torch.cuda.set_device(0)
    W_, K = args.warmup, args.steps
    L = w.L
    frames = [torch.from_numpy(f).cuda().reshape(-1) for f in w.frames(W_ + K)]
    cap = 1 << 16
    v = Vor(L, cap)
    i32 = dict(dtype=torch.int32, device="cuda")
    ccl = torch.empty(L * L, **i32)
    labels = torch.empty(L * L, **i32)
    comp = [dict(cx=torch.empty(cap, dtype=torch.float64, device="cuda"), cy=torch.empty(cap, dtype=torch.float64, device="cuda"),
                 sx=torch.empty(cap, **i32), sy=torch.empty(cap, **i32), size=torch.empty(cap, **i32),
                 root=torch.empty(cap, **i32), n=torch.zeros(1, **i32)) for _ in range(2)]
    p2n, n2p = torch.empty(cap, **i32), torch.empty(cap, **i32)
    cap_e = 8 * cap
    edges = [torch.empty(cap_e, dtype=torch.int64, device="cuda") for _ in range(2)]
    n_edges = [torch.zeros(1, dtype=torch.int64, device="cuda") for _ in range(2)]
    created, destroyed = torch.empty(cap_e, dtype=torch.int64, device="cuda"), torch.empty(cap_e, dtype=torch.int64, device="cuda")
    n_c, n_d = torch.zeros(1, dtype=torch.int64, device="cuda"), torch.zeros(1, dtype=torch.int64, device="cuda")
    stream = torch.cuda.current_stream()
    names = ["threshold_ccl", "centroids", "match", "build_cells", "label", "edges", "diff"]
    R = int(w.match_radius_cells * W.FP_ONE)
    kn = [0, 0]

    def step(i, ev=None):
        now, prv = i & 1, 1 - (i & 1)
        c, pc = comp[now], comp[prv]
        rec = (lambda j: ev[j].record(stream)) if ev else (lambda j: None)
        rec(0); v.field_threshold_ccl(frames[i], w.threshold, True, ccl)
        rec(1); v.field_centroids(ccl, w.min_size, c["cx"], c["cy"], c["sx"], c["sy"], c["size"], c["root"], c["n"])
        rec(2)
        if i > 0:
            v.match_sites(pc["sx"], pc["sy"], pc["n"], c["sx"], c["sy"], c["n"], R, p2n, n2p)
        kn[now] = int(c["n"].item())               # vor_build_cells takes n_sites on the host: one sync per frame
        rec(3); v.vor_build_cells(c["sx"][:kn[now]], c["sy"][:kn[now]])
        rec(4); v.vor_label(labels)
        rec(5); v.vor_edges(labels, edges[now], n_edges[now])
        rec(6)
        if i > 0:
            v.vor_diff(edges[prv], n_edges[prv], edges[now], n_edges[now], created, destroyed, n_c, n_d,
                       p2n=p2n, n2p=n2p, n_prev_labels=max(kn[prv], 1), n_now_labels=max(kn[now], 1))
        rec(7)

    for i in range(W_):
        step(i)
    v.vor_sync_status()
    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(8)] for _ in range(K)]
    sampler = ClockSampler(0)
    torch.cuda.synchronize()
    sampler.start()
    l0 = v.vor_launch_count()
    t0 = time.perf_counter()
    for k in range(K):
        step(W_ + k, evs[k])
    torch.cuda.synchronize()
    secs = time.perf_counter() - t0
    clocks = sampler.stop()
    launches = v.vor_launch_count() - l0
    v.vor_sync_status()
    kernel_ms = {nm: float(np.mean([evs[k][j].elapsed_time(evs[k][j + 1]) for k in range(K)])) for j, nm in enumerate(names)}
    hbm_peak, peak_src, _ = peaks()
    cells = L * L
    def roof(ms, nbytes, what):
        return {"bound": "hbm", "achieved": nbytes / (ms * 1e-3) / 1e9, "peak": hbm_peak, "unit": "GB/s",
                "frac": nbytes / (ms * 1e-3) / 1e9 / hbm_peak, "algorithmic": what, "peak_source": peak_src}
    out = {"metric": METRIC, "value": K * cells / secs, "unit": UNIT, "n_gpus": 1, "steps": K, "warmup": W_,
           "ms_per_step": 1e3 * secs / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
           "dtype": "int32", "data": "synthetic",
           "config": {"workload": w.name, "L": L, "components": kn[(W_ + K - 1) & 1], "frames": K,
                      "timing": "wall clock around K frames (one host sync per frame for the component count)"},
           "frames_per_s": K / secs, "kernel_ms": kernel_ms,
           "counts": {"n_edges": int(n_edges[(W_ + K - 1) & 1].item()), "n_created": int(n_c.item()), "n_destroyed": int(n_d.item())},
           "roofline": dict(roof(kernel_ms["threshold_ccl"], 8.0 * cells, "4 B/cell field read + 4 B/cell label written"),
                            kernel="field_threshold_ccl (3 kernels)"),
           "rooflines_other": {"field_centroids": roof(kernel_ms["centroids"], 4.0 * cells, "4 B/cell read")},
           "clocks": clocks, "gpu_launches": int(launches)}
    print(json.dumps(out), flush=True)
    v.close()


def main():
    args = parse()
    w = get_workload(args.workload)
    if isinstance(w, W.FieldWorkload):
        if args.impl == "reference" or args.gpus != 1:
            raise SystemExit("field workloads: --impl ours --gpus 1 only")
        run_field(args, w)
    elif args.impl == "reference":
        run_reference(args, w)
    else:
        run_ours(args, w)


if __name__ == "__main__":
    main()
