#!/usr/bin/env python
"""bench.py -- throughput of the batched Hough track-finding hot path on B200 (contract: see DESIGN.md "Measurement").

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--cfg 3] [--events E]
    python bench.py --gpus N                      # N > 1 without a launcher: bench.py starts the N ranks itself (torchrun)
    python bench.py --gpus N --scaling strong     # one batch cut over the ranks by hit count (default: weak, own events per rank)
    python bench.py --all-configs [--out FILE]    # one JSON line per BASELINE config 0, 1, 2 and per cell of the config-4 sweep

A "step" is one pass of the whole hot path (hough_find_clusters + hough_assign_hits) over one batch of synthetic events
of BASELINE.json's high-pile-up config (configs[3]: 100,000 events, ~2,784 hits each, 512 x 512 accumulator).  One JSON
line is printed by rank 0.  `value` is events/s with inputs resident in HBM; `e2e` the same through hough_run_host with
pinned HOST buffers (copies inside the timed region); `roofline` compares the vote rate of the fused vote+cluster kernel
with the conflict-free shared-memory atomic rate measured live on the same GPU; `cpu_baseline` is the CPU oracle
(oracle/, test infrastructure) timed on a bounded sample.  `--impl reference` times that oracle alone.
"""
from __future__ import annotations

import argparse
import json
import multiprocessing as mp
import os
import statistics
import subprocess
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2511_02742_b200 import synth  # noqa: E402  (inputs only)

METRIC = "events_per_s"
UNIT = "events/s"


def env_int(name, dflt):
    try:
        return int(os.environ.get(name, dflt))
    except ValueError:
        return dflt


def _gen_chunk(args):
    wl, chunk = args
    b = synth.generate_chunk(wl, chunk)
    return b.u, b.v, b.offsets


def generate_parallel(wl, n_events, procs):
    """First n_events events of a workload; whole chunks are generated in worker processes (seeded per chunk)."""
    n_chunks = (n_events + synth.CHUNK_EVENTS - 1) // synth.CHUNK_EVENTS
    jobs = [(wl, c) for c in range(n_chunks)]
    if procs > 1 and n_chunks > 1:
        with mp.get_context("fork").Pool(min(procs, n_chunks)) as pool:
            parts = pool.map(_gen_chunk, jobs, chunksize=1)
    else:
        parts = [_gen_chunk(j) for j in jobs]
    u = np.concatenate([p[0] for p in parts])
    v = np.concatenate([p[1] for p in parts])
    offs = [np.zeros(1, np.int64)]
    base = 0
    for p in parts:
        offs.append(p[2][1:] + base)
        base += int(p[2][-1])
    offsets = np.concatenate(offs)
    if n_events < len(offsets) - 1:
        offsets = offsets[: n_events + 1]
        u, v = u[: offsets[-1]], v[: offsets[-1]]
    return np.ascontiguousarray(u), np.ascontiguousarray(v), np.ascontiguousarray(offsets)


def oracle_params(wl):
    from oracle import hough_def as D
    return D.Params(n_theta=wl.n_theta, n_rho=wl.n_rho, rho_min=wl.rho_min, rho_max=wl.rho_max, coord_max=wl.coord_max,
                    vote_threshold=wl.vote_threshold, assign_window=wl.assign_window, max_candidates=wl.max_candidates,
                    hit_frac_bits=wl.hit_frac_bits, acc_frac_bits=-1)


def config_of(wl, n_events, n_hits, extra=None):
    c = {"workload": wl.name, "events": int(n_events), "hits": int(n_hits), "hits_per_event": round(n_hits / max(1, n_events), 1),
         "n_theta": wl.n_theta, "n_rho": wl.n_rho, "vote_threshold": wl.vote_threshold, "max_candidates": wl.max_candidates,
         "assign_window_bins": wl.assign_window_bins, "count_dtype": wl.count_dtype,
         "l2": "inputs larger than L2 (hit arrays %.2f GB)" % (n_hits * 8 / 1e9)}
    if extra:
        c.update(extra)
    return c


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md recipe)."""
    Q = "clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown," \
        "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"

    def __init__(self, index):
        self.index = index
        self.proc = None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "20",
                                          "-i", str(self.index)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except OSError:
            self.proc = None

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            out, _ = self.proc.communicate(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
            out, _ = self.proc.communicate()
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in out.splitlines():
            f = [x.strip() for x in line.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1])); pw.append(float(f[2]))
            except ValueError:
                continue
            for n, val in zip(names, f[3:7]):
                if val.lower().startswith("active"):
                    reasons.add(n)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        return {"sm_mhz": statistics.median(sm), "sm_max_mhz": max(mx), "power_w_max": max(pw), "samples": len(sm),
                "reasons": sorted(reasons)}


def time_oracle(wl, u, v, offsets, e0, n):
    """Oracle (plain C, one thread) on events [e0, e0 + n) of the batch: (seconds, outputs)."""
    from oracle import hough_c as C
    a, z = int(offsets[e0]), int(offsets[e0 + n])
    su, sv, so = u[a:z], v[a:z], offsets[e0:e0 + n + 1] - a
    t0 = time.perf_counter()
    out = C.run_batch(su, sv, so, oracle_params(wl))
    return time.perf_counter() - t0, out


def cpu_model():
    try:
        for line in open("/proc/cpuinfo"):
            if line.startswith("model name"):
                return line.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


def run_reference(args):
    """--impl reference: the CPU oracle as it stands, one thread, each step a bounded sample of the workload."""
    rank = env_int("RANK", 0)
    if rank != 0:
        return 0
    from oracle import hough_c as C
    C.build()
    wl = synth.workload(args.cfg)
    n_sample = args.ref_events
    n_total = min(wl.n_events, n_sample * (args.steps + args.warmup))
    n_total = max(n_total, n_sample)
    u, v, offsets = generate_parallel(wl, n_total, procs=min(8, os.cpu_count() or 1))
    n_avail = len(offsets) - 1
    times = []
    for s in range(args.warmup + args.steps):
        e0 = (s * n_sample) % max(1, n_avail - n_sample + 1)
        dt, _ = time_oracle(wl, u, v, offsets, e0, n_sample)
        if s >= args.warmup:
            times.append(dt)
    total = sum(times)
    value = n_sample * len(times) / total
    hits_per_event = float(offsets[-1]) / n_avail
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * total / len(times), "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "int32", "data": "synthetic",
            "votes_per_s": value * hits_per_event * wl.n_theta,
            "config": config_of(wl, wl.n_events, int(hits_per_event * wl.n_events),
                                {"sample": f"{n_sample} events per step, contiguous ranges of the first {n_avail} events"}),
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "cpu": cpu_model(),
                             "sample": f"{n_sample} events per step x {len(times)} steps, oracle/hough_oracle.c single thread"},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)
    return 0


def run_ours(args, cfg=None, hits_idx=None, grid_idx=None, quiet=False):
    """One workload on this rank's GPU; rank 0 returns (and, unless quiet, prints) the JSON line."""
    rank, world, local_rank = env_int("RANK", 0), env_int("WORLD_SIZE", 1), env_int("LOCAL_RANK", 0)
    wl = synth.workload(args.cfg if cfg is None else cfg, args.hits_idx if hits_idx is None else hits_idx,
                        args.grid_idx if grid_idx is None else grid_idx)
    strong = world > 1 and args.scaling == "strong"
    if world > 1 and not strong:
        import dataclasses
        wl = dataclasses.replace(wl, cell=wl.cell + 16 * rank)       # weak scaling: every rank gets its own events (own RNG stream)
    n_events = min(args.events or wl.n_events, wl.n_events)
    if args.max_hits and wl.hits_per_event_nominal * n_events > args.max_hits:
        n_events = max(1000, int(args.max_hits // wl.hits_per_event_nominal) // 1000 * 1000)
    procs = max(1, (os.cpu_count() or 1) // max(1, env_int("LOCAL_WORLD_SIZE", world)))
    t_gen = time.perf_counter()
    u, v, offsets = generate_parallel(wl, n_events, procs=min(procs, 32))    # before CUDA is initialised (fork)
    t_gen = time.perf_counter() - t_gen
    shard_ranges = None
    if strong:
        # strong scaling: ONE batch, cut into contiguous event ranges balanced by hit count; no collective on the data path
        from paper_2511_02742_b200 import shard
        shard_ranges = shard.shard_events(offsets, world)
        u, v, offsets = shard.local_batch(u, v, offsets, shard_ranges[rank])
        u, v = np.ascontiguousarray(u), np.ascontiguousarray(v)
        n_events = len(offsets) - 1
    n_hits = int(offsets[-1])
    max_hpe = int(np.diff(offsets).max()) if n_events else 1

    import torch
    from paper_2511_02742_b200 import hough as H
    from paper_2511_02742_b200 import build as hough_build
    try:
        hough_build.build()                                        # no-op unless libhough.so is missing or older than its sources
    except Exception as exc:  # noqa: BLE001  (no nvcc: the load below then says what is missing)
        print(f"bench.py: libhough.so was not (re)built: {exc}", file=sys.stderr)    # (every rank: the output is replaced atomically)
    H.load_library()                                               # raises if libhough.so is not built: no fallback
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)

    def barrier():
        if dist is not None:
            dist.barrier(device_ids=[local_rank])

    def max_over_ranks(x):
        if dist is None:
            return x
        t = torch.tensor([x], dtype=torch.float64, device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        return float(t.item())

    def sum_over_ranks(x):
        if dist is None:
            return x
        t = torch.tensor([x], dtype=torch.float64, device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.SUM)
        return float(t.item())

    plan = H.plan_for_workload(wl, n_events, n_hits, max_hpe, device=local_rank)
    info = H.hough_plan_query(plan)[0]
    hu, hv, ho = torch.from_numpy(u).pin_memory(), torch.from_numpy(v).pin_memory(), torch.from_numpy(offsets).pin_memory()
    du, dv, do = hu.to(dev), hv.to(dev), ho.to(dev)
    cands = torch.zeros((n_events, plan.K, H.CANDIDATE_WORDS), dtype=torch.int32, device=dev)
    n_found = torch.zeros(n_events, dtype=torch.int32, device=dev)
    labels = torch.empty(n_hits, dtype=torch.int32, device=dev)
    stream = torch.cuda.current_stream(dev)

    def step(ev=None):
        if ev is not None:
            ev[0].record(stream)
        H.hough_find_clusters(plan, du, dv, do, cands, n_found, stream=stream)
        if ev is not None:
            ev[1].record(stream)
        H.hough_assign_hits(plan, du, dv, do, cands, n_found, labels, stream=stream)
        if ev is not None:
            ev[2].record(stream)

    for _ in range(args.warmup):
        step()
    torch.cuda.synchronize(dev)
    status = H.hough_plan_status(plan)

    # ---- timed region: device-resident inputs
    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(args.steps)]
    sampler = ClockSampler(local_rank)
    sampler.start()
    time.sleep(0.15)
    launches0 = H.hough_plan_launch_count(plan)
    barrier()
    torch.cuda.synchronize(dev)
    e_begin, e_end = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e_begin.record(stream)
    for s in range(args.steps):
        step(evs[s])
    e_end.record(stream)
    torch.cuda.synchronize(dev)
    barrier()
    launches = H.hough_plan_launch_count(plan) - launches0
    clocks = sampler.stop()
    deferred = int(H.hough_plan_debug_counters(plan)[15])          # events the fast kernel handed to the general kernel (last step)
    ms_total = max_over_ranks(e_begin.elapsed_time(e_end))
    ms_step = ms_total / args.steps
    ms_find = statistics.mean(e[0].elapsed_time(e[1]) for e in evs)
    ms_assign = statistics.mean(e[1].elapsed_time(e[2]) for e in evs)
    step_ms = [e[0].elapsed_time(e[2]) for e in evs]
    events_all = sum_over_ranks(float(n_events))
    hits_all = sum_over_ranks(float(n_hits))
    value = events_all / (ms_step * 1e-3)
    votes_per_s = hits_all * wl.n_theta / (ms_step * 1e-3)

    # ---- end to end through hough_run_host: pinned host buffers, copies inside the timed region
    e2e = None
    if not args.no_e2e:
        hc = torch.zeros((n_events, plan.K, H.CANDIDATE_WORDS), dtype=torch.int32).pin_memory()
        hn = torch.zeros(n_events, dtype=torch.int32).pin_memory()
        hl = torch.zeros(n_hits, dtype=torch.int32).pin_memory()
        n_e2e_warm, n_e2e = min(args.warmup, 3), max(3, min(args.steps, 5))
        for _ in range(n_e2e_warm):
            H.hough_run_host(plan, hu, hv, ho, hc, hn, hl)
        barrier()
        torch.cuda.synchronize(dev)
        t0 = time.perf_counter()
        for _ in range(n_e2e):
            H.hough_run_host(plan, hu, hv, ho, hc, hn, hl)         # synchronises before it returns
        t_e2e = max_over_ranks(time.perf_counter() - t0) / n_e2e
        barrier()
        e2e = {"value": events_all / t_e2e, "unit": UNIT, "ms_per_step": t_e2e * 1e3, "steps": n_e2e,
               "h2d_bytes_per_step": int(n_hits * 8 + (n_events + 1) * 8),
               "d2h_bytes_per_step": int(n_hits * 4 + n_events * plan.K * 32 + n_events * 4),
               "same_as_device_results": bool((hn == n_found.cpu()).all().item() and (hl == labels.cpu()).all().item())}
        del hc, hl

    gathered = None
    if strong:
        # per-event results back in event order on every rank (NCCL all-gather; outside the timed region: the data path has no collective)
        from paper_2511_02742_b200 import shard
        gathered = shard.gather_per_event(n_found, shard_ranges)
        assert gathered.numel() == sum(b - a for a, b in shard_ranges)

    line = None
    if rank == 0:
        # ---- roofline of the dominant kernel (fused vote + peak/cluster finding): shared-memory atomic adds
        peak_ops, peak_mhz = H.hough_measure_smem_atomic_peak(local_rank, 50.0)
        votes_launch = float(n_hits) * wl.n_theta
        achieved = votes_launch / (ms_find * 1e-3)
        hbm_bytes = n_hits * 8 + (n_events + 1) * 8 + n_events * 4 + float(torch.clamp(n_found, max=plan.K).sum().item()) * 32
        peaks_file = os.path.join(ROOT, "MEASURED_PEAKS.json")
        hbm_peak = json.load(open(peaks_file)).get("hbm_gbs") if os.path.exists(peaks_file) else None
        sm_max = (clocks.get("sm_max_mhz") or 1965.0) * 1e6
        # diagnostic second ceiling: a vote needs at least 5 issued instructions (2 IMAD, SHF, LOP3, RED) on 4 schedulers / SM
        alu_peak = info["n_sm"] * 4 * sm_max / 5.0 * 32
        roofline = {"bound": "smem_atomic",
                    "kernel": ("hough_fast_kernel (hough_find_clusters)" if info["fast_groups"] and 2 * deferred <= n_events else
                               "hough_event_kernel (hough_find_clusters; %d of %d events)" % (deferred if info["fast_groups"] else n_events, n_events)),
                    "achieved": achieved / 1e9, "peak": peak_ops / 1e9, "unit": "Gatomic/s", "frac": achieved / peak_ops,
                    "peak_source": "hough_measure_smem_atomic_peak, measured live on this GPU (nothing but conflict-free "
                                   "red.shared.add.u32, %.0f MHz); MEASURED_PEAKS.json has no shared-memory figure" % peak_mhz,
                    "alu_issue": {"peak": alu_peak / 1e9, "unit": "Gvote/s", "frac": achieved / alu_peak,
                                  "note": "5 issue slots per vote x 4 schedulers x n_sm x sm_max_mhz (DESIGN.md)"},
                    "ms_per_launch": ms_find, "share_of_step": ms_find / (ms_find + ms_assign),
                    # the reported fraction of the whole pipeline (find + assign) next to the dominant kernel's
                    "frac_pipeline": votes_launch / ((ms_find + ms_assign) * 1e-3) / peak_ops,
                    # second, diagnostic ceiling for sparse workloads: every tile byte is zeroed and scanned once per event
                    # at 128 B / clk / SM of shared-memory bandwidth (u16 or i32 counters as the plan chose)
                    "dense_tile": dense_tile_ceiling(info, wl, sm_max, n_events / (ms_find * 1e-3)),
                    "traffic": traffic_from_profiles(wl.name, "hough_fast_kernel" if info["fast_groups"] else "hough_event_kernel")
                    if n_events == wl.n_events else None,
                    "hbm": {"algorithmic_bytes": hbm_bytes, "achieved_gbs": hbm_bytes / (ms_find * 1e-3) / 1e9,
                            "peak_gbs": hbm_peak, "peak_source": "MEASURED_PEAKS.json" if hbm_peak else "absent",
                            "frac": (hbm_bytes / (ms_find * 1e-3) / 1e9 / hbm_peak) if hbm_peak else None}}
        # ---- CPU baseline: the oracle as it stands, one thread, bounded sample; doubles as a parity spot check
        cpu = None
        if world == 1 and not args.no_cpu_baseline:
            ns = min(args.cpu_events, n_events)
            dt, out = time_oracle(wl, u, v, offsets, 0, ns)
            k = plan.K
            gc = H.candidates_to_numpy(cands[:ns])
            same = bool((out["n_found"] == n_found[:ns].cpu().numpy()).all()
                        and (out["labels"] == labels[: int(offsets[ns])].cpu().numpy()).all()
                        and all(gc[e, :min(int(out["n_found"][e]), k)].tobytes() == out["cands"][e, :min(int(out["n_found"][e]), k)].tobytes()
                                for e in range(ns)))
            cpu = {"value": ns / dt, "unit": UNIT, "cores": 1, "kind": "oracle", "cpu": cpu_model(), "host_cores": os.cpu_count(),
                   "sample": f"first {ns} events of the workload, {dt:.1f} s, oracle/hough_oracle.c single thread",
                   "gpu_outputs_identical_on_sample": same}
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
                "ms_per_step": ms_step, "higher_is_better": True, "scaling": "strong" if strong else "weak", "vs_baseline": None,
                "dtype": "int32",
                "data": "synthetic", "votes_per_s": votes_per_s,
                "config": config_of(wl, int(events_all) if strong else n_events, int(hits_all) if strong else n_hits,
                                    {"parallelism": (f"one batch cut into {world} contiguous event ranges balanced by hit count "
                                                     "(shard.shard_events), no collective on the data path; per-event results "
                                                     "all-gathered afterwards" if strong else
                                                     f"events sharded over {world} GPU(s), no collective"),
                                     "plan": info, "status_word": status, "deferred_events": deferred, "gen_s": round(t_gen, 1)}),
                "kernel_ms": {"hough_find_clusters": ms_find, "hough_assign_hits": ms_assign},
                "ms_per_step_median": statistics.median(step_ms), "ms_per_step_best": min(step_ms),     # this rank's steps
                "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches), "roofline": roofline, "cpu_baseline": cpu}
    H.hough_plan_destroy(plan)
    if dist is not None:
        dist.destroy_process_group()
    if line is not None and not quiet:
        print(json.dumps(line), flush=True)
    return line


def traffic_from_profiles(workload, kernel):
    """dram__bytes_read.sum + dram__bytes_write.sum of one launch of `kernel` on `workload`, read from the committed ncu table
    profiles/ncu_traffic.csv (one row per `ncu --set full` capture; the newest row wins); None if no capture exists."""
    path = os.path.join(ROOT, "profiles", "ncu_traffic.csv")
    best = None
    try:
        with open(path) as f:
            header = f.readline().strip().split(",")
            for row in f:
                r = dict(zip(header, row.strip().split(",")))
                if r.get("workload") == workload and r.get("kernel", "").startswith(kernel):
                    best = int(r["dram_bytes_read"]) + int(r["dram_bytes_write"])
    except (OSError, ValueError, KeyError):
        return None
    return best


def dense_tile_ceiling(info, wl, sm_hz, events_per_s):
    tile_bytes = wl.n_theta * wl.n_rho * (2 if info["fast_groups"] else info["counter_bytes"])
    peak = info["n_sm"] * sm_hz * 128.0 / (2.0 * tile_bytes)
    return {"peak_events_per_s": peak, "frac": events_per_s / peak, "tile_bytes_per_event": tile_bytes}


ALL_CONFIGS = [(0, 0, 0), (1, 0, 0), (2, 0, 0)] + [(4, h, g) for h in range(4) for g in range(4)]


def run_all_configs(args):
    """One JSON line per BASELINE config 0, 1, 2 and per cell of the config-4 roofline sweep, written to
    --out; the default bench line (config 3) is not part of this mode.  Single GPU."""
    if env_int("WORLD_SIZE", 1) != 1:
        print("bench.py --all-configs runs on one GPU", file=sys.stderr)
        return 2
    out = args.out or os.path.join(ROOT, "gpurun_out", "all_configs.jsonl")
    os.makedirs(os.path.dirname(out), exist_ok=True)
    args.no_e2e = True
    args.cpu_events = min(args.cpu_events, 64)
    n = 0
    with open(out, "w") as f:
        for cfg, h, g in ALL_CONFIGS:
            line = run_ours(args, cfg, h, g, quiet=True)
            f.write(json.dumps(line) + "\n")
            f.flush()
            n += 1
    print(json.dumps({"all_configs": n, "out": out}), flush=True)
    return 0


def free_port():
    import socket
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def launch_ranks(args):
    """`python bench.py --gpus N` without a launcher: start the N ranks with torchrun on this node and wait for them."""
    import torch
    have = torch.cuda.device_count()
    if have < args.gpus:
        print(f"bench.py --gpus {args.gpus}: only {have} CUDA device(s) visible", file=sys.stderr)
        return 2
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}", "--master-addr", "127.0.0.1",
           "--master-port", str(free_port()), os.path.abspath(__file__)] + sys.argv[1:]
    return subprocess.call(cmd)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--cfg", type=int, default=3, help="BASELINE.json config index (default: 3, the high-pile-up config)")
    ap.add_argument("--hits-idx", type=int, default=0, help="config 4: index into hits/event {100,500,2000,8000}")
    ap.add_argument("--grid-idx", type=int, default=0, help="config 4: index into grids {128,256,512,1024}")
    ap.add_argument("--events", type=int, default=0, help="use only the first E events (debugging; not a bench value)")
    ap.add_argument("--cpu-events", type=int, default=1500, help="events of the cpu_baseline sample")
    ap.add_argument("--ref-events", type=int, default=200, help="--impl reference: events per step")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--scaling", default="weak", choices=["weak", "strong"], help="N > 1: own events per rank, or one batch cut over the ranks")
    ap.add_argument("--all-configs", action="store_true", help="configs 0, 1, 2 and the 16 cells of config 4, one JSON line each, to --out")
    ap.add_argument("--out", default="", help="--all-configs: output file (default gpurun_out/all_configs.jsonl)")
    ap.add_argument("--max-hits", type=float, default=0, help="cap a workload at about this many hits (fewer events; recorded in config)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.impl == "reference":
        return run_reference(args)
    world_env = os.environ.get("WORLD_SIZE")
    if world_env is None and args.gpus > 1:
        return launch_ranks(args)                                      # no launcher: start the ranks ourselves
    if int(world_env or 1) != args.gpus:
        print(f"bench.py: --gpus {args.gpus} but WORLD_SIZE={world_env or 1}: launch one rank per GPU (or drop the launcher and let "
              "bench.py start them)", file=sys.stderr)
        return 2
    if args.all_configs:
        return run_all_configs(args)
    run_ours(args)
    return 0


if __name__ == "__main__":
    sys.exit(main())
