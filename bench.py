#!/usr/bin/env python
"""Benchmark of the Phase-I TPC sector tracker (BASELINE.json: TPC clusters/s, sector tracking, device-timed, 1 B200).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 3] [--impl ours|reference]

A step = one pass of the whole hot path (K1..K6, tpc_track_sectors) over one synthetic event of
BASELINE.json:configs[--config] (default 3 = central Pb-Pb, the config the target is quoted on) that is already
resident in HBM.  The L2 is flushed (256 MiB write) before every timed step, outside the CUDA-event bracket.
N > 1: one process per GPU (torchrun), each rank tracks its own event (seed = rank) - events are independent
(PAPER.md:82), no collective on the data path, weak scaling; time = max over ranks.
`--impl reference` times the CPU oracle (oracle/) on the host cores instead; see DESIGN.md "Measurement".
Prints ONE JSON line on rank 0.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "tpc_clusters_per_sec_sector_tracking"
UNIT = "clusters/s"
# Algorithmic HBM bytes per kernel: N clusters, B bins, S start hits,
# H = sum of tracklet hits, T tracks, C clusters in tracks.


def algorithmic_bytes(st: dict) -> dict:
    n, s, h = st["n_clusters"], st["n_start_hits"], st["n_tracklet_hits"]
    t, c = st["n_tracks"], st["n_track_clusters"]
    return {
        "K1_sort_grid": 8 * n + 8 * n + 4 * n + 4 * n + 4 * n,       # in y,z; out (y,z), orig, binStart(~N), weight=0
        "K2_neighbours": 8 * n + 4 * n + 8 * n,                      # hits once, bins once, links out
        "K3K4_clean_start": 8 * n + 8 * n + 16 * s,                  # raw links in, cleaned out, start list (16 B each)
        "K5_construct": 28 * h + 4 * h + 128 * s,                    # per row step: link/bin 12 + hit 8 + cand 8; rowHit; record
        "K6a_weights": 4 * h + 8 * h + 32 * s,                       # rowHit in, atomicMax rmw, record header
        "K6b_select": 4 * h + 4 * h + 128 * s + 8 * c + 112 * t,     # rowHit, weight, record; orig + ids out, tracks out
    }


def source_sha16() -> str:
    """Hash of the CUDA sources the library is built from: ties profiles/kernel_counters.json to a build."""
    import hashlib
    h = hashlib.sha256()
    d = os.path.join(ROOT, "paper_1712_09430_b200", "csrc")
    for f in sorted(os.listdir(d)):
        if f.endswith((".cu", ".cuh")):
            h.update(open(os.path.join(d, f), "rb").read())
    return h.hexdigest()[:16]


COUNTERS = os.path.join(ROOT, "profiles", "kernel_counters.json")
NCU_KERNELS = {"K1_sort_grid": "k1_sort_grid", "K2_neighbours": "k2_neighbours", "K3K4_clean_start": "k3_clean_start",
               "K5_construct": "k5_construct_phased", "K6a_weights": "k6_weights", "K6b_select": "k6_select"}


def ncu_summary(rep: str):
    """`bench.py --ncu-summary REPORT.ncu-rep`: per-kernel counters of one `ncu --set full` capture of bench.py ->
    profiles/kernel_counters.json (instructions, DRAM bytes, lanes per instruction), stamped with the hash of the CUDA
    sources.  bench.py quotes them (roofline.traffic, roofline_issue) only while that hash is the current one."""
    import csv
    import subprocess
    raw = subprocess.run(["ncu", "-i", rep, "--page", "raw", "--csv"], capture_output=True, text=True, check=True).stdout
    rows = list(csv.reader(raw.splitlines()))
    hdr = rows[0]
    col = {h: i for i, h in enumerate(hdr)}
    units = rows[1]
    out = {"source_sha16": source_sha16(), "report": os.path.basename(rep), "kernels": {}}
    for key, name in NCU_KERNELS.items():
        for r in rows[2:]:
            if name in r[col["Kernel Name"]]:
                def val(m, scale_bytes=False):
                    v = float(r[col[m]].replace(",", ""))
                    if scale_bytes:
                        v *= {"byte": 1, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9}[units[col[m]]]
                    return v
                out["kernels"][key] = {
                    "inst_executed": int(val("smsp__inst_executed.sum")),
                    "threads_per_inst": round(val("smsp__thread_inst_executed_per_inst_executed.ratio"), 2),
                    "dram_bytes": int(val("dram__bytes_read.sum", True) + val("dram__bytes_write.sum", True)),
                    "ncu_us": round(val("gpu__time_duration.sum"), 2),
                    "warps_per_scheduler": round(val("smsp__warps_active.avg.per_cycle_active"), 2),
                }
                break
    json.dump(out, open(COUNTERS, "w"), indent=1)
    print(json.dumps(out))


def kernel_counters():
    """profiles/kernel_counters.json if it describes the current sources, else None (never a stale number)."""
    try:
        c = json.load(open(COUNTERS))
        return c if c.get("source_sha16") == source_sha16() else None
    except Exception:
        return None


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index: int):
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self._stop = threading.Event()
        self._thr = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = int(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
        except Exception:
            self.nv = None

    def _run(self):
        nv = self.nv
        names = {"hw_slowdown": 0x8, "sw_power_cap": 0x4, "hw_thermal_slowdown": 0x40, "sw_thermal_slowdown": 0x20,
                 "hw_power_brake_slowdown": 0x80}
        while not self._stop.is_set():
            try:
                self.samples.append(int(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
                try:
                    r = int(nv.nvmlDeviceGetCurrentClocksEventReasons(self.h))
                except Exception:
                    r = int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h))
                for k, bit in names.items():
                    if r & bit:
                        self.reasons.add(k)
            except Exception:
                pass
            time.sleep(0.002)

    def start(self):
        if self.nv is not None:
            self._thr = threading.Thread(target=self._run, daemon=True)
            self._thr.start()

    def stop(self):
        self._stop.set()
        if self._thr:
            self._thr.join()
        s = sorted(self.samples)
        return {"sm_mhz": (s[len(s) // 2] if s else None), "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "samples": len(s)}


def init_dist(n_gpus: int):
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    dist = None
    if world > 1:
        import torch
        import torch.distributed as dist_
        backend = "nccl" if torch.cuda.is_available() else "gloo"
        if backend == "nccl":
            torch.cuda.set_device(local)
        dist_.init_process_group(backend=backend)
        dist = dist_
    return rank, world, local, dist


def reduce_over_ranks(dist, value: float, op: str, device) -> float:
    """max / sum of a python float over all ranks (no-op for world size 1)."""
    if dist is None:
        return value
    import torch
    t = torch.tensor([value], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX if op == "max" else dist.ReduceOp.SUM)
    return float(t.item())


def aggregate(dist, device, n_clusters_rank: int, step_ms_rank: float):
    """Whole-job throughput: all ranks' clusters / the slowest rank's time (weak scaling, no data-path collective)."""
    n_total = reduce_over_ranks(dist, float(n_clusters_rank), "sum", device)
    ms = reduce_over_ranks(dist, step_ms_rank, "max", device)
    return n_total / (ms * 1e-3), ms, int(n_total)


def oracle_baseline(ev, budget_s: float = 15.0):
    """cpu_baseline leg: the oracle as it stands, single-threaded, on a bounded sample of the same workload."""
    import oracle
    # probe one sector to size the sample
    t0 = time.perf_counter()
    sub = ev.sector_slice(0)
    oracle.Oracle(1, ev.n_rows, ev.row_x, ev.bz).run(sub.row_counts, sub.y, sub.z, fetch=False)
    t_sector = max(time.perf_counter() - t0, 1e-4)
    n_sec = int(max(1, min(ev.n_sectors, budget_s / t_sector)))
    if n_sec >= ev.n_sectors:
        sample, desc = ev, f"whole event ({ev.n_clusters} clusters), best of 2 runs"
        runs = 2 if 2 * t_sector * ev.n_sectors < 2 * budget_s else 1
    else:
        import datagen
        b = ev.row_base
        hi = int(b[n_sec * ev.n_rows])
        sample = datagen.Event(n_sec, ev.n_rows, ev.row_x, ev.bz, ev.row_counts[:n_sec].copy(), ev.y[:hi], ev.z[:hi],
                               ev.truth[:hi])
        desc, runs = f"sectors 0..{n_sec - 1} of the event ({hi} clusters), 1 run", 1
    o = oracle.Oracle(sample.n_sectors, sample.n_rows, sample.row_x, sample.bz)
    best = 1e30
    for _ in range(runs):
        t0 = time.perf_counter()
        o.run(sample.row_counts, sample.y, sample.z, fetch=False)
        best = min(best, time.perf_counter() - t0)
    out = {"value": sample.n_clusters / best, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": desc,
           "seconds": best, "stage_seconds": o.stage_seconds()}
    # north_star: decisions the oracle's own candidates tie within 1e-6 relative are "counted and reported"
    res = o.fetch()
    out["near_ties"] = {"s2_hits": int(res.tie_s2.sum()), "tracklets": int(res.tracklets["near_tie"].sum()),
                        "of_hits": int(res.n_clusters), "of_tracklets": int(res.tracklets.size)}
    # the SAME single-threaded oracle, one instance per sector, on a pool of P host
    # threads (sectors are independent; ctypes releases the GIL).  Context next to the 1-core number.
    try:
        from concurrent.futures import ThreadPoolExecutor
        p = len(os.sched_getaffinity(0))
        subs = [sample.sector_slice(s) for s in range(sample.n_sectors)]
        if p > 1 and len(subs) > 1:
            def one(sub):
                oracle.Oracle(1, sub.n_rows, sub.row_x, sub.bz).run(sub.row_counts, sub.y, sub.z, fetch=False)
            with ThreadPoolExecutor(max_workers=p) as ex:
                t0 = time.perf_counter()
                list(ex.map(one, subs))
                dt = time.perf_counter() - t0
            out["all_cores"] = {"value": sample.n_clusters / dt, "unit": UNIT, "cores": min(p, len(subs)),
                                "seconds": dt, "how": "one oracle instance per sector on a thread pool"}
    except Exception as e:      # the 1-core number is the contract; this one is context
        out["all_cores"] = {"error": str(e)}
    return out


def multi_event_leg(torch, binding, datagen, args, params, dev, rank: int, k: int, reps: int):
    """Several events per call (one event cannot fill the GPU; two tracker instances per GPU gave
    -24 % per event there).  Phase-I sectors are independent, so k events are loaded as 36*k sectors of
    ONE tracker and tracked by one tpc_track_sectors call: every kernel then works on k events at once.
    Same timing rules as the main leg (inputs resident in HBM, L2 flushed before every call, CUDA events)."""
    evs = [datagen.config_event(args.config, seed=1000 + rank * k + i) for i in range(k)]
    e0 = evs[0]
    counts = np.concatenate([e.row_counts.reshape(-1) for e in evs]).reshape(e0.n_sectors * k, e0.n_rows)
    n_total = int(sum(e.n_clusters for e in evs))
    trk = binding.Tracker(e0.n_sectors * k, e0.n_rows, e0.row_x, e0.bz, params)
    stream = torch.cuda.current_stream()
    trk.set_stream(stream.cuda_stream)
    trk.allocate_workspace(n_total, device=dev)
    y = torch.from_numpy(np.concatenate([e.y for e in evs])).to(dev)
    z = torch.from_numpy(np.concatenate([e.z for e in evs])).to(dev)
    trk.load_event(counts, y, z)
    trk.set_output_prefetch(False)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    times = []
    for i in range(3 + reps):
        flush.fill_(1)
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(stream)
        trk.track_sectors()
        b.record(stream)
        trk.sync()
        if i >= 3:
            times.append(a.elapsed_time(b))
    ms = sum(times) / len(times)
    trk.set_kernel_timing(True)                  # one more call with the events between the kernels, for the table only
    flush.fill_(1)
    trk.track_sectors()
    trk.sync()
    st = trk.get_stats()
    trk.destroy()
    return {"events_per_call": k, "calls": reps, "n_clusters_per_call": n_total, "ms_per_call": ms, "ms_per_event": ms / k,
            "value": n_total / (ms * 1e-3), "unit": UNIT, "n_tracks": st["n_tracks"],
            "kernel_us_per_event": {kk: round(v / k, 1) for kk, v in st["kernel_us"].items()},
            "note": "k independent synthetic events (other seeds) as 36*k sectors of one tracker, one call"}


def instances_leg(torch, binding, ev, params, dev, n_inst: int, n_events: int):
    """PAPER.md:82-84 (several tracker instances share the GPU; the paper measures -24 % per event with two): n_inst
    trackers on n_inst streams, inputs resident in HBM, ONE host thread issuing tpc_track_sectors round robin and
    waiting for the oldest; wall clock per event.  Extra key, not the metric (no L2 flush: the instances' 0.4 GB
    workspaces evict each other)."""
    pipes = []
    for _ in range(n_inst):
        sti = torch.cuda.Stream(device=dev)
        ti = binding.Tracker(ev.n_sectors, ev.n_rows, ev.row_x, ev.bz, params)
        ti.set_stream(sti.cuda_stream)
        ti.allocate_workspace(ev.n_clusters, device=dev)
        ti.set_output_prefetch(False)
        y, z = torch.from_numpy(ev.y).to(dev), torch.from_numpy(ev.z).to(dev)
        ti.load_event(ev.row_counts, y, z)
        pipes.append((ti, sti, y, z))

    def run(n):
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        for i in range(n + n_inst):
            ti = pipes[i % n_inst][0]
            if i >= n_inst:
                ti.sync()
            if i < n:
                ti.track_sectors()
        torch.cuda.synchronize()
        return (time.perf_counter() - t0) / n * 1e3
    run(2 * n_inst)
    ms = run(n_events)
    for p_ in pipes:
        p_[0].destroy()
    return ms


def time_frame_leg(torch, binding, datagen, params, dev, reps: int = 3):
    """BASELINE.json:configs[4] (extra key, not the headline): a Run-3-style time frame - 20 overlapped central events,
    ~31.6 M clusters - tracked by ONE tpc_track_sectors call (north_star).  Same timing rules as the main leg."""
    ev = datagen.config_event(4, seed=0)
    trk = binding.Tracker(ev.n_sectors, ev.n_rows, ev.row_x, ev.bz, params)
    stream = torch.cuda.current_stream()
    trk.set_stream(stream.cuda_stream)
    ws = trk.allocate_workspace(ev.n_clusters, device=dev)
    trk.load_event(ev.row_counts, torch.from_numpy(ev.y).to(dev), torch.from_numpy(ev.z).to(dev))
    trk.set_output_prefetch(False)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    times = []
    for i in range(1 + reps):
        flush.fill_(1)
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(stream)
        trk.track_sectors()
        b.record(stream)
        trk.sync()
        if i >= 1:
            times.append(a.elapsed_time(b))
    ms = sum(times) / len(times)
    trk.set_kernel_timing(True)
    flush.fill_(1)
    trk.track_sectors()
    trk.sync()
    st = trk.get_stats()
    trk.destroy()
    # the same time frame in slices of 9 sectors through a quarter of the workspace (tpc_track_event_sliced:
    # synchronous, results of every slice downloaded - wall clock of the call, input resident on the device)
    per_sector = ev.row_counts.reshape(ev.n_sectors, ev.n_rows).sum(axis=1)
    fullest = max(int(per_sector[s:s + 9].sum()) for s in range(0, ev.n_sectors, 9))
    trk = binding.Tracker(ev.n_sectors, ev.n_rows, ev.row_x, ev.bz, params)
    trk.set_stream(stream.cuda_stream)
    ws_sl = trk.allocate_workspace(fullest, device=dev)
    dy, dz = torch.from_numpy(ev.y).to(dev), torch.from_numpy(ev.z).to(dev)
    trk.track_event_sliced(ev.row_counts, dy, dz, 9)
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    tr_sl, _ = trk.track_event_sliced(ev.row_counts, dy, dz, 9)
    sliced_ms = (time.perf_counter() - t0) * 1e3
    trk.destroy()
    sliced = {"sectors_per_slice": 9, "ms_per_call_wall_with_download": round(sliced_ms, 2), "n_tracks": int(tr_sl.size),
              "workspace_bytes": int(ws_sl), "workspace_over_whole": round(ws_sl / ws, 3)}
    return {"workload": "config4:timeframe-20x-central", "n_clusters": ev.n_clusters, "calls": reps, "ms_per_call": ms, "sliced": sliced,
            "value": ev.n_clusters / (ms * 1e-3), "unit": UNIT, "central_events_per_sec": 20.0 / (ms * 1e-3),
            "n_start_hits": st["n_start_hits"], "n_tracklet_hits": st["n_tracklet_hits"], "n_tracks": st["n_tracks"],
            "workspace_over_input": round(ws / (12.0 * ev.n_clusters), 2),
            "kernel_us": {k: round(v, 1) for k, v in st["kernel_us"].items()}}


def run_reference(args, rank, world, dist):
    """--impl reference: the CPU oracle, timed on the host cores, same metric/config (rank 0 only)."""
    if rank != 0:
        return
    import datagen
    import oracle
    ev = datagen.config_event(args.config, seed=0)
    # bounded sample: keep (steps+warmup) * t_step within ~2.5 minutes
    t0 = time.perf_counter()
    sub = ev.sector_slice(0)
    oracle.Oracle(1, ev.n_rows, ev.row_x, ev.bz).run(sub.row_counts, sub.y, sub.z, fetch=False)
    t_sector = max(time.perf_counter() - t0, 1e-4)
    n_sec = int(max(1, min(ev.n_sectors, 150.0 / ((args.steps + args.warmup) * t_sector))))
    b = ev.row_base
    hi = int(b[n_sec * ev.n_rows])
    sample = datagen.Event(n_sec, ev.n_rows, ev.row_x, ev.bz, ev.row_counts[:n_sec].copy(), ev.y[:hi], ev.z[:hi], ev.truth[:hi])
    o = oracle.Oracle(n_sec, ev.n_rows, ev.row_x, ev.bz)
    for _ in range(args.warmup):
        o.run(sample.row_counts, sample.y, sample.z, fetch=False)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        o.run(sample.row_counts, sample.y, sample.z, fetch=False)
    dt = (time.perf_counter() - t0) / args.steps
    val = sample.n_clusters / dt
    desc = f"sectors 0..{n_sec - 1} of config {args.config} ({hi} of {ev.n_clusters} clusters) per step"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": dt * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": f"config{args.config}:{datagen.CONFIG_NAMES[args.config]}", "sample": desc},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": desc},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=30)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--config", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--e2e-instances", type=int, default=6, help="tracker instances (streams) the ONE host thread of the end-to-end leg keeps in flight")
    ap.add_argument("--neighbour-staging", action="store_true", help="K2 with its neighbour rows staged in shared memory (tpc_set_neighbour_staging; slower, for the ncu comparison)")
    ap.add_argument("--no-time-frame", action="store_true", help="skip the configs[4] leg (20 overlapped central events in one call)")
    ap.add_argument("--ncu-summary", default=None, metavar="REPORT.ncu-rep",
                    help="no benchmark: extract per-kernel counters of an ncu capture of bench.py into profiles/kernel_counters.json")
    ap.add_argument("--bins-per-hit", type=float, default=None, help="override tpc_params.grid_bins_per_hit (tuning)")
    ap.add_argument("--events-per-call", type=int, default=4,
                    help="extra leg: this many events tracked by one call (PAPER.md:82-84); 0 or 1 = skip")
    args = ap.parse_args()
    if args.ncu_summary:
        ncu_summary(args.ncu_summary)
        return
    rank, world, local, dist = init_dist(args.gpus)
    if args.impl == "reference":
        run_reference(args, rank, world, dist)
        if dist is not None:
            dist.barrier()
            dist.destroy_process_group()
        return

    import torch
    import datagen
    from paper_1712_09430_b200 import binding
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    dev = torch.device("cuda", local)
    torch.cuda.set_device(dev)
    warmup = max(args.warmup, 3)

    ev = datagen.config_event(args.config, seed=rank)
    params = binding.default_params()
    if args.bins_per_hit is not None:
        params.grid_bins_per_hit = args.bins_per_hit
    trk = binding.Tracker(ev.n_sectors, ev.n_rows, ev.row_x, ev.bz, params)
    stream = torch.cuda.current_stream()
    trk.set_stream(stream.cuda_stream)
    ws_bytes = trk.allocate_workspace(ev.n_clusters, device=dev)
    y_dev, z_dev = torch.from_numpy(ev.y).to(dev), torch.from_numpy(ev.z).to(dev)
    trk.load_event(ev.row_counts, y_dev, z_dev)          # inputs resident in HBM before the timed region
    trk.set_output_prefetch(False)                       # device-timed leg: K1..K6 only (no result download queued behind K6)
    trk.set_neighbour_staging(args.neighbour_staging)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)

    def step_device():
        flush.fill_(1)                                  # evict the 126 MB L2 (outside the event bracket)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        trk.track_sectors()
        e1.record(stream)
        return e0, e1

    # warm-up: at least W steps and at least ~0.3 s of load so the clocks are up
    t0 = time.perf_counter()
    n_warm = 0
    while n_warm < warmup or time.perf_counter() - t0 < 0.3:
        step_device()
        n_warm += 1
        if n_warm % 8 == 0:
            torch.cuda.synchronize()
    torch.cuda.synchronize()
    if dist is not None:
        dist.barrier()
    sampler = ClockSampler(local)
    sampler.start()
    torch.cuda.synchronize()
    # timed region: K steps as a user runs them (no CUDA events between the kernels: tpctrk.h tpc_set_kernel_timing)
    events = []
    for _ in range(args.steps):
        events.append(step_device())
        trk.sync()
    torch.cuda.synchronize()
    if dist is not None:
        dist.barrier()
    step_ms = sum(a.elapsed_time(b) for a, b in events) / args.steps
    # the same K steps again with an event between the kernels: per-kernel times for the roofline / kernel table
    # (the five extra event records cost ~14 us per step, reported as ms_per_step_kernel_timing)
    trk.set_kernel_timing(True)
    events, kern = [], {k: 0.0 for k in binding.KERNEL_NAMES}
    for _ in range(args.steps):
        events.append(step_device())
        trk.sync()                                       # per-kernel device times of this step
        st = trk.get_stats()
        for k, v in st["kernel_us"].items():
            kern[k] += v
    torch.cuda.synchronize()
    clocks = sampler.stop()
    step_ms_timing = sum(a.elapsed_time(b) for a, b in events) / args.steps
    trk.set_kernel_timing(False)
    kern = {k: v / args.steps for k, v in kern.items()}
    st = trk.get_stats()
    value, ms, n_total = aggregate(dist, dev, ev.n_clusters, step_ms)

    # ---- Phase II: track merging (K7) and final fit (K8, next-2); extra key, not part of the
    # metric: device times of tpc_merge_tracks / tpc_refit_tracks on the tracks of this event, L2 flushed before, CUDA events inside the library
    merge_us, refit_us = [], []
    for _ in range(max(3, min(args.steps, 10))):
        flush.fill_(1)
        trk.track_sectors()
        trk.merge_tracks()
        trk.refit_tracks()
        trk.get_merged()
        trk.get_refit()
        merge_us.append(trk.get_stats()["merge_us"])
        refit_us.append(trk.get_stats()["refit_us"])
    stm = trk.get_stats()
    merge_leg = {"kernel": "K7 track merging (tpc_merge_tracks: 7 launches)", "us": round(sum(merge_us[1:]) / len(merge_us[1:]), 1),
                 "n_tracks": stm["n_tracks"], "n_links": stm["n_merge_links"], "n_merged_tracks": stm["n_merged_tracks"],
                 "refit_kernel": "K8 final fit of the merged tracks (tpc_refit_tracks: 1 launch)",
                 "refit_us": round(sum(refit_us[1:]) / len(refit_us[1:]), 1)}

    # ---- end to end through the C ABI with HOST buffers (pinned), H2D + D2H of every step inside the timed region.
    # ONE host thread keeps n_pipe tracker instances (each on its own stream) in flight, round robin: for the oldest
    # instance tpc_get_tracks (waits once: the download was queued behind its kernels), then
    # tpc_load_event (page-locked input, returns when the copy is queued) and tpc_track_sectors for its next event -
    # the paper's DMA || kernels pipeline (Fig. 4) with several tracker instances per GPU.
    n_pipe = max(1, args.e2e_instances)
    pipes = []
    for i in range(n_pipe):
        sti = torch.cuda.Stream(device=dev)
        ti = binding.Tracker(ev.n_sectors, ev.n_rows, ev.row_x, ev.bz, params)
        ti.set_stream(sti.cuda_stream)
        ti.allocate_workspace(ev.n_clusters, device=dev)
        pipes.append((ti, sti, torch.from_numpy(ev.y.copy()).pin_memory(), torch.from_numpy(ev.z.copy()).pin_memory()))
    last = [None]

    def e2e_run(n_events):
        """n_events events through the n_pipe instances; returns wall seconds."""
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        for i in range(n_events + n_pipe):
            ti, _, yp, zp = pipes[i % n_pipe]
            if i >= n_pipe:
                last[0] = ti.get_tracks(copy=False)          # result of event i - n_pipe
            if i < n_events:
                ti.load_event(ev.row_counts, yp.numpy(), zp.numpy())
                ti.track_sectors()
        torch.cuda.synchronize()
        return time.perf_counter() - t0

    e2e_run(2 * n_pipe)
    if dist is not None:
        dist.barrier()
    n_e2e = max(12, min(4 * args.steps, 96)) // n_pipe * n_pipe
    e2e_ms = e2e_run(n_e2e) / n_e2e * 1e3
    tr, ids = last[0]
    e2e_value, e2e_ms_max, _ = aggregate(dist, dev, ev.n_clusters, e2e_ms)
    h2d = 8 * ev.n_clusters + 48 * ev.n_sectors * ev.n_rows + 4 * (ev.n_sectors + 1)
    est_t, est_c = int(tr.shape[0]) + int(tr.shape[0]) // 4 + 64, int(ids.shape[0]) + int(ids.shape[0]) // 4 + 1024
    d2h = 112 * est_t + 4 * min(est_c, ev.n_clusters) + 64           # what is queued: the estimate (counts + 25 %), not the exact size
    e2e_refetches = sum(p[0].get_stats()["n_output_refetches"] for p in pipes)
    for p_ in pipes:
        p_[0].destroy()

    # ---- roofline of the dominant kernel + per-kernel table
    peak, peak_src = measured_peaks()
    ab = algorithmic_bytes(st)
    if st.get("k6a_fused"):
        # the phased K5 kernel ran the K6a weights pass itself: its bytes are K5's, K6a's launch returned at once
        ab["K5_construct"] += ab["K6a_weights"]
        ab["K6a_weights"] = 0
    dom = max(kern, key=kern.get)
    per_kernel = {k: {"us": round(kern[k], 2), "alg_bytes": ab[k], "gbs": round(ab[k] / (kern[k] * 1e-6) / 1e9, 1),
                      "frac": round(ab[k] / (kern[k] * 1e-6) / 1e9 / peak, 4)} for k in kern}
    achieved = ab[dom] / (kern[dom] * 1e-6) / 1e9
    # counters of an ncu capture of THIS build (profiles/kernel_counters.json carries the hash of the CUDA sources;
    # with other sources the file is ignored: no stale number)
    cnt = kernel_counters()
    traffic = cnt["kernels"].get(dom, {}).get("dram_bytes") if cnt else None
    # What bounds these kernels is instruction issue and latency, not HBM: issue roofline =
    # warp instructions executed (ncu smsp__inst_executed.sum of the same build) / CUDA-event time, against the peak of
    # one instruction per cycle and scheduler: SMs x 4 x the SM clock sampled during the timed region.
    roof_issue = None
    if cnt and clocks.get("sm_mhz"):
        sms = torch.cuda.get_device_properties(dev).multi_processor_count
        peak_ips = sms * 4 * clocks["sm_mhz"] * 1e6
        roof_issue = {"unit": "warp-inst/s", "peak": peak_ips, "peak_source": f"{sms} SMs x 4 schedulers x {clocks['sm_mhz']} MHz (sampled)",
                      "counters": "profiles/kernel_counters.json (ncu, same CUDA sources)", "kernels": {}}
        for k in kern:
            c = cnt["kernels"].get(k)
            if c and kern[k] > 0:
                roof_issue["kernels"][k] = {"inst": c["inst_executed"], "frac": round(c["inst_executed"] / (kern[k] * 1e-6) / peak_ips, 4),
                                            "threads_per_inst": c["threads_per_inst"], "warps_per_scheduler": c["warps_per_scheduler"]}
    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "warmup_actual": n_warm, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic",
        "config": {"workload": f"config{args.config}:{datagen.CONFIG_NAMES[args.config]}", "n_clusters_per_gpu": ev.n_clusters,
                   "n_clusters_total": n_total, "events_per_sec": world / (ms * 1e-3), "seed": "rank", "l2": "flushed (256 MiB write) before every timed step",
                   "parallelism": "one event per GPU, no collective" if world > 1 else "single GPU",
                   "n_start_hits": st["n_start_hits"], "n_tracklet_hits": st["n_tracklet_hits"], "n_tracks": st["n_tracks"],
                   "workspace_bytes": ws_bytes, "workspace_over_input": round(ws_bytes / (12.0 * ev.n_clusters), 2),
                   "grid_bins_per_hit": float(params.grid_bins_per_hit),
                   "k6a_fused_into_k5": bool(st.get("k6a_fused")),
                   "ms_per_step_kernel_timing": step_ms_timing,
                   "kernel_times": "second pass of the same K steps with a CUDA event between the kernels (tpc_set_kernel_timing)"},
        "clocks": clocks,
        "e2e": {"value": e2e_value, "unit": UNIT, "ms_per_step": e2e_ms_max, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                "steps": n_e2e, "output_refetches": e2e_refetches,
                "pipeline": f"one host thread, {n_pipe} tracker instances (streams) in flight: page-locked input read by DMA without blocking, result download queued behind K6 (estimate = last counts + 25 %), one wait per event"},
        "gpu_launches": 2 * args.steps * trk.launches_per_track(),      # the K timed steps and their second pass with kernel timing
        "roofline": {"bound": "hbm", "kernel": dom, "achieved": round(achieved, 2), "peak": peak, "unit": "GB/s",
                     "frac": round(achieved / peak, 5), "traffic": traffic, "peak_source": peak_src,
                     "frac_of_8TBs_nominal": round(achieved / 8000.0, 5),
                     "whole_step": {"alg_bytes": sum(ab.values()), "gbs": round(sum(ab.values()) / (ms * 1e-3) / 1e9, 1),
                                    "frac": round(sum(ab.values()) / (ms * 1e-3) / 1e9 / peak, 5)}},
        "kernels": per_kernel,
    }
    if roof_issue:
        out["roofline_issue"] = roof_issue
    out["merge"] = merge_leg
    if args.events_per_call > 1 and args.config <= 3:
        me = multi_event_leg(torch, binding, datagen, args, params, dev, rank, args.events_per_call, max(3, min(args.steps, 10)))
        me["value"] = reduce_over_ranks(dist, me["value"], "sum", dev)      # whole job: sum of the ranks' rates
        out["multi_event"] = me
    if rank == 0 and args.events_per_call > 1 and args.config <= 3:
        n_ev = max(12, min(4 * args.steps, 48))
        one = instances_leg(torch, binding, ev, params, dev, 1, n_ev)
        n_inst = max(2, args.e2e_instances)
        three = instances_leg(torch, binding, ev, params, dev, n_inst, n_ev // n_inst * n_inst)
        out["concurrent_instances"] = {"instances": n_inst, "ms_per_event": round(three, 4), "one_instance_ms_per_event": round(one, 4),
                                       "value": ev.n_clusters / (three * 1e-3), "unit": UNIT,
                                       "note": "PAPER.md:82-84: trackers on separate streams, inputs resident, no L2 flush, wall clock"}
    if rank == 0 and not args.no_time_frame and args.config == 3:
        del trk, y_dev, z_dev                            # (the time frame needs ~9 GB of workspace)
        out["time_frame"] = time_frame_leg(torch, binding, datagen, params, dev)
    if rank == 0 and not args.no_cpu_baseline:
        out["cpu_baseline"] = oracle_baseline(datagen.config_event(args.config, seed=0))
        out["config"]["near_ties"] = out["cpu_baseline"].get("near_ties")
    if dist is not None:
        dist.barrier()
    if rank == 0:
        print(json.dumps(out), flush=True)
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
