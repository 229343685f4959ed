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

# Per-launch ncu figures of the committed `ncu --set full` capture (config 5 only): DRAM bytes read + written,
# issue-slot utilisation, warp instructions.  profiles/r3_traffic.md names the command that produced the table.
# These figures are REPLAYED from that committed capture, never measured by a bench run: every object that carries
# them says so ("measured_in_this_run": false) and names the file and the commit the capture was taken from.
NCU_TABLE_REL = "profiles/r3_traffic.csv"
NCU_TABLE = os.path.join(ROOT, *NCU_TABLE_REL.split("/"))
NCU_TABLE_COMMIT = "55183a2"     # the kernels in the table are unchanged since (label / edges / diff kernels)


def ncu_table():
    """kernel name -> dict of floats; {} when the table is missing."""
    out = {}
    if os.path.exists(NCU_TABLE):
        import csv
        with open(NCU_TABLE) as f:
            for row in csv.DictReader(f):
                out[row["kernel"]] = {k: float(v) for k, v in row.items() if k != "kernel" and v not in ("", None)}
    return out


def ncu_for(table, name):
    """ncu row of the kernel whose name starts like `name` (template arguments are spelled differently)."""
    base = name.split("<")[0]
    for k, v in table.items():
        if k.split("<")[0] == base:
            return v
    return {}


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
    ap.add_argument("--shard", default="sequences", choices=["sequences", "strips"],
                    help="N > 1: independent sequences per rank (default, weak scaling) or row strips of ONE lattice "
                         "(strong scaling: strips.py, one all-gather + merge per frame)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-field-leg", action="store_true", help="skip the short config-4 field-path leg of the default line")
    ap.add_argument("--cpu-sample-L", type=int, default=0,
                    help="lattice side of the oracle's sample (0 = the full workload, in both arms)")
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
def oracle_frame_seconds(w, frames, threads=0):
    """Time the oracle, as it stands, on `frames` (list of (sx, sy)); returns (seconds, cells).
    threads: OpenMP threads of the labelling (0 = all the process may use); edges and diff are serial."""
    import oracle
    prev = np.empty(0, np.uint64)
    t0 = time.perf_counter()
    for sx, sy in frames:
        lab = oracle.label_cells(w.L, sx, sy, w.bucket_cells, threads)
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
    Ls = args.cpu_sample_L or w.L                   # the FULL workload (config 5: ~4.3 s per frame on 16 cores)
    ws = w if Ls == w.L else W.scaled(5, Ls) if w.kind == "jittered_grid" else w
    frames = list(ws.frames(args.warmup + args.steps))
    for sx, sy in frames[:args.warmup]:
        oracle.edges(oracle.label_cells(ws.L, sx, sy, ws.bucket_cells))
    secs, cells = oracle_frame_seconds(ws, frames[args.warmup:])
    cores = oracle.num_threads()
    val = cells / secs
    sample = (f"{args.steps} frames of {ws.name} ({ws.L}^2 cells, {ws.n_sites} sites"
              + ("" if ws.L == w.L else f": same density and structure as {w.name}")
              + f"); label_cells on {cores} threads, edges + diff on 1 (serial in the oracle)")
    out = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
           "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * secs / args.steps,
           "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "int64",
           "data": "synthetic", "config": {"workload": w.name, "L": w.L, "n_sites": w.n_sites,
                                           "sample_L": ws.L, "sample_sites": ws.n_sites},
           "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample,
                            "threads": {"label_cells": cores, "edges": 1, "diff": 1}},
           "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
           "gpu_launches": 0}
    print(json.dumps(out), flush=True)


# ------------------------------------------------------------------------------------------ our arm
def frame_algorithmic_bytes(cells, n_sites, e_prev, e_now, n_c, n_d):
    """What one site-driven frame must move: the label image written (a2) and read (a3),
    the edge list written (a4) and both lists read by the comparison (a5), the flip lists written, and the
    cell list (about 40 B per site)."""
    return 8.0 * cells + 8.0 * e_now + 8.0 * (e_prev + e_now) + 8.0 * (n_c + n_d) + 40.0 * n_sites


def run_ours(args, w):
    import torch
    import torch.distributed as dist
    from paper_1607_00908_b200.binding import Vor

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world != args.gpus:
        raise SystemExit(f"bench.py: --gpus {args.gpus} but WORLD_SIZE={world}")
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
    row_ptr = [torch.zeros(n + 1, dtype=torch.int32, device="cuda") for _ in range(2)]
    created = torch.empty(cap_e, dtype=torch.int64, device="cuda")
    destroyed = torch.empty(cap_e, dtype=torch.int64, device="cuda")
    n_c = torch.zeros(1, dtype=torch.int64, device="cuda")
    n_d = torch.zeros(1, dtype=torch.int64, device="cuda")
    stream = torch.cuda.current_stream()
    names = ["build_cells", "label", "edges", "diff"]

    # One step = a1..a5 through the C ABI: cell list, labels, edge list with its row offsets (the
    # compressed adjacency matrix), row-by-row comparison with the previous frame's list.
    def step(i, ev=None):
        now, prev = i & 1, 1 - (i & 1)
        sx, sy = dframes[i]
        if ev: ev[0].record(stream)
        v.vor_build_cells(sx, sy)
        if ev: ev[1].record(stream)
        v.vor_label(labels)
        if ev: ev[2].record(stream)
        v.vor_edges_rows(labels, edges[now], n_edges[now], row_ptr[now])
        if ev: ev[3].record(stream)
        v.vor_diff_rows(edges[prev], row_ptr[prev], edges[now], row_ptr[now], n, created, destroyed, n_c, n_d)
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
    last = (W_ + K - 1) & 1
    counts = {"n_edges": int(n_edges[last].item()), "n_edges_prev": int(n_edges[1 - last].item()),
              "n_created": int(n_c.item()), "n_destroyed": int(n_d.item())}
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
    # couples of active vertices, breaking / arising class, T1 partner
    t1_keys, t1_partner = torch.empty(cap_e, dtype=torch.int64, device="cuda"), torch.empty(cap_e, dtype=torch.int64, device="cuda")
    t1_cls, t1_cp, t1_cn = (torch.empty(cap_e, **i32) for _ in range(3))
    t1_n = torch.zeros(1, dtype=torch.int64, device="cuda")
    def t1():
        v.vor_t1_events(edges[1 - last], n_edges[1 - last], edges[last], n_edges[last], created, n_c, destroyed, n_d,
                        ev_bufs[0], t1_keys, t1_cls, t1_cp, t1_cn, t1_partner, t1_n)
    for _ in range(3):
        t1()
    e0.record(stream)
    for _ in range(10):
        t1()
    e1.record(stream)
    torch.cuda.synchronize()
    k_ = int(t1_n.item())
    events_info["t1"] = {"ms": e0.elapsed_time(e1) / 10, "couples": k_,
                         "breaking": int((t1_cls[:k_] == 1).sum().item()), "arising": int((t1_cls[:k_] == 2).sum().item()),
                         "t1_quadruples": int(((t1_cls[:k_] == 1) & (t1_partner[:k_] != -1)).sum().item()),
                         "api": "vor_t1_events: couples, breaking / arising, common neighbours, T1 partner (PAPER.md:238, 248-266)"}
    del t1_keys, t1_partner, t1_cls, t1_cp, t1_cn

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
    v.close()
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    hbm_peak, peak_src, sm_max_mhz = peaks()
    is_cfg5 = wr.name.startswith("cfg5_throughput_stress")
    ncu = ncu_table() if is_cfg5 else {}

    # every kernel is reported against the measured HBM copy rate with ITS algorithmic
    # bytes; `traffic` = DRAM bytes of one launch REPLAYED from the committed ncu capture (config 5 only;
    # `traffic_source` says so); `achieved`, `frac` and `launch_ms` are measured live by this run.
    def hbm_roof(name, nbytes, what, ms=None):
        if ms is None:
            if name not in kernel_launch_ms:
                return None
            ms = kernel_launch_ms[name]
        t = ncu_for(ncu, name)
        r = {"kernel": name, "bound": "hbm", "achieved": nbytes / (ms * 1e-3) / 1e9, "peak": hbm_peak, "unit": "GB/s",
             "frac": nbytes / (ms * 1e-3) / 1e9 / hbm_peak, "traffic": t.get("dram_bytes"), "launch_ms": ms,
             "algorithmic": what, "peak_source": peak_src}
        if t:
            replayed = {"measured_in_this_run": False, "source": NCU_TABLE_REL, "capture_commit": NCU_TABLE_COMMIT}
            r["traffic_source"] = replayed
            r["ncu"] = {"issue_active_pct": t.get("issue_active_pct"), "warp_inst_per_cell":
                        t["warp_inst"] / cells_per_step if "warp_inst" in t else None, **replayed}
        return r

    # The dominant kernel is the labelling kernel (one launch per step).  Its §8(d) unit is the 4 B/cell it
    # writes; what actually limits it is integer issue (the nested ncu figures: issue slots busy, warp
    # instructions per cell), which only fewer instructions can improve.
    lab_name = max((nm for nm in kernel_launch_ms if "label" in nm), key=lambda nm: kernel_launch_ms[nm])
    roofline = hbm_roof(lab_name, 4.0 * cells_per_step, "4 B/cell label write")
    roofline["limited_by"] = "integer issue slots, not HBM (DESIGN.md 5.2, 5.9)"
    ne, nep = counts["n_edges"], counts["n_edges_prev"]
    ncd = counts["n_created"] + counts["n_destroyed"]
    diff_ms = sum(kernel_launch_ms.get(k, 0.0) for k in ("diff_rows_mark_kernel", "diff_rows_write_kernel"))
    others = {
        "edges_stream_kernel": hbm_roof("edges_stream_kernel", 4.0 * cells_per_step, "4 B/cell label read"),
        "vor_diff_rows (mark + write)": hbm_roof(
            "diff_rows", 8.0 * (ne + nep) + 8.0 * ncd + 8.0 * n,
            "8 B x (E_prev + E_now) read + 8 B x (created + destroyed) written + 2 x 4 B/site row offsets; "
            "L2-resident", ms=diff_ms) if diff_ms > 0 else None,
        "vor_edges_rows (stream + insert + finish)": hbm_roof(
            "vor_edges_rows", edges_bytes(cells_per_step, ne), "4 B/cell label read + 8 B/edge written",
            ms=kernel_ms["edges"]),
    }
    frame_bytes = frame_algorithmic_bytes(cells_per_step, n, nep, ne, counts["n_created"], counts["n_destroyed"])
    step_s = ms_total / K * 1e-3
    frame_roofline = {"bound": "hbm", "achieved": frame_bytes / step_s / 1e9, "peak": hbm_peak, "unit": "GB/s",
                      "frac": frame_bytes / step_s / 1e9 / hbm_peak, "algorithmic_bytes_per_frame": frame_bytes,
                      "algorithmic": "label image written + read, edge list written, both lists read by the "
                                     "comparison, flip lists written, 40 B/site cell list",
                      "peak_source": peak_src}
    if e2e:
        frame_roofline["e2e_frac"] = frame_bytes / (e2e["ms_per_step"] * 1e-3) / 1e9 / hbm_peak
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
        "frame_roofline": frame_roofline,
        "events": events_info,
        "clocks": clocks, "gpu_launches": int(launches),
    }
    if e2e:
        out["e2e"] = e2e
    if not args.no_field_leg and world == 1 and is_cfg5:
        out["field_path"] = field_leg(W.config(4), 2, 4)
    if not args.no_cpu_baseline and world == 1:
        import oracle
        Ls = args.cpu_sample_L or w.L
        ws = w if Ls == w.L else W.scaled(5, Ls)
        fr = list(ws.frames(1))
        secs, cells = oracle_frame_seconds(ws, fr)
        nt = oracle.num_threads()
        out["cpu_baseline"] = {"value": cells / secs, "unit": UNIT, "cores": nt, "kind": "oracle",
                               "threads": {"label_cells": nt, "edges": 1, "diff": 1},
                               "sample": f"1 frame of {ws.name} ({ws.L}^2 cells, {ws.n_sites} sites): label_cells on "
                                         f"{nt} threads, edges + diff on 1 (serial in the oracle), {secs:.1f} s"}
        # the same oracle on ONE thread, on a 1/16-area copy of the workload
        w1 = W.scaled(5, max(256, ws.L // 4)) if ws.kind == "jittered_grid" and ws.L >= 1024 else ws
        s1, c1 = oracle_frame_seconds(w1, list(w1.frames(1)), threads=1)
        out["cpu_baseline"]["single_thread"] = {
            "value": c1 / s1, "unit": UNIT, "cores": 1,
            "sample": f"1 frame of {w1.name} ({w1.L}^2 cells, {w1.n_sites} sites), {s1:.1f} s"}
    print(json.dumps(out), flush=True)
    if world > 1:
        dist.destroy_process_group()


# ------------------------------------------------------------------------------------------ field path
FIELD_GROUPS = (("threshold_ccl", ("ccl_",)), ("centroids", ("comp_", "accumulate", "centroid")),
                ("match", ("match_",)), ("build_cells", ("count_sites", "scan_", "scatter_sites")),
                ("label", ("label_",)), ("edges", ("edges_", "rows_insert")),
                ("diff", ("translate_", "filter_", "sort_unique", "diff_", "maps_")))


def field_group(kernel_name: str) -> str:
    kernel_name = kernel_name.strip("()")
    for g, prefixes in FIELD_GROUPS:
        if any(kernel_name.startswith(p) for p in prefixes):
            return g
    return "other"


def field_leg(w, warmup: int, steps: int):
    """Frames of a field-derived workload (config 3 or 4) through field_frame_device: rows a6..a8 then a1..a5
    chained on the device without a host synchronisation (the bubble count stays in a device scalar).
    Returns per-frame time (CUDA events around the K frames), per-kernel launch times from a second pass
    and the §8(d) fractions of the field kernels."""
    import torch
    from paper_1607_00908_b200.binding import Vor
    L = w.L
    frames = [torch.from_numpy(f).cuda().reshape(-1) for f in w.frames(warmup + steps)]
    v = Vor(L, 1 << 16)
    R = int(w.match_radius_cells * W.FP_ONE)
    stream = torch.cuda.current_stream()

    def step(i):
        v.field_frame_device(frames[i], w.threshold, True, w.min_size, R)

    for i in range(warmup):
        step(i)
    v.vor_sync_status()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    l0 = v.vor_launch_count()
    e0.record(stream)
    for k in range(steps):
        step(warmup + k)
    e1.record(stream)
    torch.cuda.synchronize()
    launches = v.vor_launch_count() - l0
    ms = e0.elapsed_time(e1) / steps
    counts_host = v.vor_download(v.field_frame_results()["counts"], np.zeros(5, np.int64))
    v.vor_profile_begin()
    for k in range(steps):
        step(warmup + k)
    prof = v.vor_profile_end()
    v.vor_sync_status()
    per_kernel, groups = {}, {}
    for nm, t in prof:
        per_kernel.setdefault(nm, []).append(t)
    kernel_launch_ms = {nm: float(np.sum(x)) / steps for nm, x in per_kernel.items()}
    for nm, t in kernel_launch_ms.items():
        groups[field_group(nm)] = groups.get(field_group(nm), 0.0) + t
    hbm_peak, peak_src, _ = peaks()
    cells = L * L

    def roof(ms_, nbytes, what):
        return {"bound": "hbm", "achieved": nbytes / (ms_ * 1e-3) / 1e9, "peak": hbm_peak, "unit": "GB/s",
                "frac": nbytes / (ms_ * 1e-3) / 1e9 / hbm_peak, "launch_ms": ms_, "algorithmic": what,
                "peak_source": peak_src}
    out = {"workload": w.name, "L": L, "frames": steps, "ms_per_frame": ms, "frames_per_s": 1e3 / ms,
           "cells_per_s": cells / (ms * 1e-3), "gpu_launches_per_frame": launches / steps,
           "api": "field_frame_device (a6 -> a7 -> a8 -> a1..a5 on the device, no host synchronisation)",
           "counts": {"bubbles": int(counts_host[0]), "n_edges": int(counts_host[1]), "n_created": int(counts_host[2]),
                      "n_destroyed": int(counts_host[3])},
           "kernel_ms": groups, "kernel_launch_ms": kernel_launch_ms,
           "rooflines": {
               "field_threshold_ccl": roof(groups.get("threshold_ccl", float("nan")), 8.0 * cells,
                                           "4 B/cell field read + 4 B/cell bubble label written"),
               "field_centroids": roof(groups.get("centroids", float("nan")), 4.0 * cells, "4 B/cell read")}}
    v.close()
    return out


def run_field(args, w):
    """--workload cfg3 | cfg4: one step = one frame of the field-derived path (rows a6..a8, then a1..a5 with
    the isomorphism).  Single GPU; not the default bench line (the metric is quoted on config 5)."""
    import torch
    torch.cuda.set_device(0)
    sampler = ClockSampler(0)
    sampler.start()
    leg = field_leg(w, args.warmup, args.steps)
    clocks = sampler.stop()
    out = {"metric": METRIC, "value": leg["cells_per_s"], "unit": UNIT, "n_gpus": 1, "steps": args.steps,
           "warmup": args.warmup, "ms_per_step": leg["ms_per_frame"], "higher_is_better": True, "scaling": "weak",
           "vs_baseline": None, "dtype": "int32", "data": "synthetic",
           "config": {"workload": w.name, "L": w.L, "components": leg["counts"]["bubbles"], "frames": args.steps,
                      "timing": "CUDA events around K frames of field_frame_device (no host synchronisation)"},
           "frames_per_s": leg["frames_per_s"], "kernel_ms": leg["kernel_ms"], "kernel_launch_ms": leg["kernel_launch_ms"],
           "counts": leg["counts"],
           "roofline": dict(leg["rooflines"]["field_threshold_ccl"], kernel="field_threshold_ccl"),
           "rooflines_other": {"field_centroids": leg["rooflines"]["field_centroids"]},
           "clocks": clocks, "gpu_launches": int(round(leg["gpu_launches_per_frame"] * args.steps))}
    print(json.dumps(out), flush=True)


def spawn_ranks(args) -> int:
    """`python bench.py --gpus N` without a launcher: start the N ranks ourselves (torch.distributed.run, one
    process per GPU, rendezvous on 127.0.0.1) and pass their output through."""
    import socket
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    env = dict(os.environ)
    env.setdefault("NCCL_DEBUG", "WARN")
    return subprocess.call(cmd, env=env)


def run_strips(args, w):
    """--shard strips: ONE lattice per step, its rows split over the ranks.  Every rank labels its
    strip (+ the next strip's first row), extracts its keys, all-gathers the lists, merges them and compares the
    merged list with the previous frame's.  value = L^2 * K / time: strong scaling."""
    import torch
    import torch.distributed as dist
    from paper_1607_00908_b200.binding import Vor
    from paper_1607_00908_b200.strips import StripFrame

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world != args.gpus:
        raise SystemExit(f"bench.py: --gpus {args.gpus} but WORLD_SIZE={world}")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    W_, K = args.warmup, args.steps
    frames = [(torch.from_numpy(sx).cuda(), torch.from_numpy(sy).cuda()) for sx, sy in w.frames(W_ + K)]   # same on every rank
    L, n = w.L, w.n_sites
    cap_e = 4 * n + 1024
    v = Vor(L, n, max(1 << 20, 16 * n, world * cap_e))
    fr = [StripFrame(v, n, cap_e, cap_e) for _ in range(2)]                # ping-pong: this frame's / the previous list
    created = torch.empty(cap_e, dtype=torch.int64, device="cuda"); destroyed = torch.empty_like(created)
    n_c = torch.zeros(1, dtype=torch.int64, device="cuda"); n_d = torch.zeros_like(n_c)
    stream = torch.cuda.current_stream()

    def step(i):
        now, prev = fr[i & 1], fr[1 - (i & 1)]
        now.compute(*frames[i])
        v.vor_diff(prev.edges, prev.n_edges, now.edges, now.n_edges, created, destroyed, n_c, n_d)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    sampler = ClockSampler(local)
    sampler.start()
    for i in range(W_):
        step(i)
    v.vor_sync_status()
    t0, t1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    l0 = v.vor_launch_count()
    t0.record(stream)
    for k in range(K):
        step(W_ + k)
    t1.record(stream)
    barrier()
    launches = v.vor_launch_count() - l0
    v.vor_sync_status()
    ms_total = reduce_max(t0.elapsed_time(t1), world, "cuda")
    v.vor_profile_begin()
    for k in range(K):
        step(W_ + k)
    per = {}
    for nm, ms in v.vor_profile_end():
        per[nm] = per.get(nm, 0.0) + ms / K
    clocks = sampler.stop()
    if rank == 0:
        print(json.dumps({"metric": METRIC, "value": L * L * K / (ms_total * 1e-3), "unit": UNIT, "n_gpus": world, "steps": K,
                          "warmup": W_, "ms_per_step": ms_total / K, "higher_is_better": True, "scaling": "strong",
                          "vs_baseline": None, "dtype": "int32", "data": "synthetic",
                          "config": {"workload": w.name, "L": L, "n_sites": n, "parallelism": f"row strips x {world}",
                                     "rows_per_rank": fr[0].rows, "l2_policy": "strip image exceeds L2"},
                          "kernel_launch_ms": per, "gpu_launches": launches, "clocks": clocks,
                          "counts": {"n_edges": int(fr[(W_ + K - 1) & 1].n_edges.item()), "n_created": int(n_c.item()),
                                     "n_destroyed": int(n_d.item())}}))
    if world > 1:
        dist.destroy_process_group()


def main():
    args = parse()
    w = get_workload(args.workload)
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        raise SystemExit(spawn_ranks(args))
    if isinstance(w, W.FieldWorkload):
        if args.impl == "reference" or args.gpus != 1:
            raise SystemExit("field workloads: --impl ours --gpus 1 only")
        run_field(args, w)
    elif args.impl == "reference":
        run_reference(args, w)
    elif args.shard == "strips":
        run_strips(args, w)
    else:
        run_ours(args, w)


if __name__ == "__main__":
    main()
