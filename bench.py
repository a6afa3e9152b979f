#!/usr/bin/env python
"""bench.py -- throughput of the TPC sector tracker on the synthetic drift-window workload.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--windows NW] [--impl ours|reference]

A "step" is one pass of the whole hot path (S1..S6, one tpc_track_sectors call) over one batch of NW CFG:4 drift
windows (BASELINE.json configs[3]/[4]: 5 overlapping Pb-Pb events per window; 36*NW independent sector instances).
`value` = clusters/s with the inputs resident in HBM; `e2e` = the same metric through tpc_track_sectors_host with
pinned HOST buffers (upload, tracking and result download inside the timed region).
N > 1 (torchrun): every rank tracks its own NW windows (weak scaling, no data-path collective).
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
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_1709_00618_b200 import datagen, sharding  # noqa: E402

METRIC = "TPC clusters/sec tracked on 1 B200 (ms/event); achieved HBM GB/s vs peak"
UNIT = "clusters/s"
# algorithmic bytes the staged method moves per cluster (whole path / S5 only)
BYTES_PER_CLUSTER_PATH = 130.0
BYTES_PER_CLUSTER_S5 = 34.0
# fp32 operations per unit of S5 work, counted from the formulas in csrc/kf_math.cuh
FLOP_TRANSPORT, FLOP_UPDATE, FLOP_EXAMINE, FLOP_SEARCH = 150.0, 93.0, 7.0, 18.0
FP32_LANES_PER_SM, N_SM = 128, 148
# ncu dram bytes per launch of the dominant kernel: read from the JSON committed next to the profile it was taken
# from (it names the commit, the workload and the cluster count); reported only when this run's workload matches.
TRAFFIC_JSON = os.path.join(ROOT, "profiles", "roofline_traffic.json")
# results the e2e runs bring back: the fitted tracks and the cluster -> track assignment (once)
E2E_WANT = ("cluster_owner", "trk_params", "trk_nhits", "trk_sector")


WORKLOAD = "cfg5"  # set from --workload before the batch is generated (module global: the worker processes fork)
WORKLOADS = {"cfg5": "CFG:4 drift windows (5 overlapping Pb-Pb-like events each)",
             "cfg3": "CFG:3 central Pb-Pb-like events (8,000 primaries + 20 % secondaries, 10 % noise)",
             "cfg2": "CFG:2 peripheral Pb-Pb-like events (1,000 primaries, 5 % noise)"}


def _gen_window(seed):
    if WORKLOAD == "cfg3":
        return datagen.central_event(seed)
    if WORKLOAD == "cfg2":
        return datagen.full_event(seed)
    return datagen.drift_window(seed)


def make_batch(n_windows, seed0, rank=0):
    """NW CFG:4 windows, generated in parallel worker processes (before CUDA is touched)."""
    seeds = sharding.window_seeds(n_windows, seed0, rank)
    n_proc = max(1, min(n_windows, (os.cpu_count() or 2) // max(1, int(os.environ.get("LOCAL_WORLD_SIZE", "1")))))
    if n_proc > 1:
        import multiprocessing as mp
        with mp.get_context("fork").Pool(n_proc) as pool:
            evs = pool.map(_gen_window, seeds)
    else:
        evs = [_gen_window(s) for s in seeds]
    return evs, datagen.concat_events(evs, name=f"cfg5_batch{n_windows}")


def shard_job(evs, batch, world, rank):
    """Strong scaling ("slice the timeframe in parts as we do with the TPC sectors"): ONE
    job, the same on every rank, cut into contiguous blocks of whole windows balanced by cluster count; rank r tracks
    its block as a self-contained input.  No data-path collective: only the small counts are gathered afterwards.
    Returns (the rank's windows, its batch, what it owns)."""
    import dataclasses
    i0, ni, c0, nc = sharding.partition_instances(batch.row_offsets, batch.n_inst, batch.n_rows, world, rank)
    cl, ro = sharding.local_problem(batch.clusters, batch.row_offsets, batch.n_rows, i0, ni)
    local = dataclasses.replace(batch, clusters=np.ascontiguousarray(cl), row_offsets=np.ascontiguousarray(ro),
                                labels=batch.labels[c0:c0 + nc], n_inst=ni, truth={},
                                name=f"{batch.name}_shard{rank}of{world}")
    return evs[i0 // 36:(i0 + ni) // 36], local, dict(inst0=i0, n_inst=ni, cluster0=c0, n_clusters=nc)


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.lines = []
        self.proc = None
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", "100", "-i", str(index)], stdout=subprocess.PIPE, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except Exception:
            self.proc = None

    def _read(self):
        for ln in self.proc.stdout:
            self.lines.append((time.time(), ln.strip()))

    def stop(self, t0, t1):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        sm, smax, reasons, power = [], None, set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        rows = [l for (ts, l) in self.lines if t0 <= ts <= t1 + 0.2] or [l for (_, l) in self.lines[-3:]]
        for l in rows:
            f = [x.strip() for x in l.split(",")]
            try:
                sm.append(float(f[0])); smax = float(f[1]); power.append(float(f[2]))
            except Exception:
                continue
            for nme, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nme)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": smax, "reasons": sorted(reasons),
                "power_w_max": max(power) if power else None, "samples": len(sm)}


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            d = json.load(f)
        return float(d["hbm_gbs"]), float(d.get("sm_max_mhz", 1965.0)), "measured (MEASURED_PEAKS.json)"
    return 6650.0, 1965.0, "fallback (B200_PROFILING.md)"


def cpu_baseline(evs, budget_windows=1):
    """The oracle as it stands, on the host cores, on a bounded sample (first windows of the batch)."""
    from oracle.tpc_oracle import Oracle
    ev = datagen.concat_events(evs[:budget_windows]) if budget_windows > 1 else evs[0]
    cores = min(os.cpu_count() or 1, ev.n_inst)
    o = Oracle.for_event(ev)
    t = time.perf_counter()
    c = o.track_count(ev.clusters, ev.row_offsets, ev.n_inst, n_threads=cores)
    dt = time.perf_counter() - t
    # the same oracle on ONE core, on one sector instance of the sample (S8d: single-threaded and all-core figures)
    R = ev.n_rows
    i_big = int(np.argmax(np.diff(ev.row_offsets[::R])))
    lo, hi = int(ev.row_offsets[i_big * R]), int(ev.row_offsets[(i_big + 1) * R])
    ro1 = (ev.row_offsets[i_big * R:(i_big + 1) * R + 1] - lo).astype(np.int32)
    t1 = time.perf_counter()
    o.track_count(ev.clusters[lo:hi], ro1, 1, n_threads=1)
    dt1 = time.perf_counter() - t1
    return {"value": ev.n_clusters / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
            "single_core_value": (hi - lo) / dt1,
            "sample": f"{budget_windows} drift window(s) of the batch, {ev.n_clusters} clusters, {ev.n_inst} sector "
                      f"instances, one OpenMP thread per instance up to all cores, {dt:.2f} s",
            "tracks": c["n_tracks"]}, dt


def run_reference(args):
    """--impl reference: the CPU oracle on the same workload recipe, each step a bounded sample (one window)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    evs, _ = make_batch(1, args.seed0)
    times = []
    info = None
    for i in range(args.warmup + args.steps):
        info, dt = cpu_baseline(evs, 1)
        if i >= args.warmup:
            times.append(dt)
    n = evs[0].n_clusters
    v = n * len(times) / sum(times)
    info["value"] = v
    line = {"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * sum(times) / len(times), "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64 (Kalman filter) / f32 (neighbour search)",
            "data": "synthetic", "config": {"workload": "cfg4_drift_window (bounded sample: 1 window per step)",
                                            "clusters_per_step": n, "seed0": args.seed0},
            "cpu_baseline": info,
            "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line))


def measure_fp32_peak(torch, dev):
    """fp32 FMA rate of this GPU from the bench-only library (csrc_bench/fp32_peak.cu: 8 independent FMA chains per
    thread, 64 warps per SM), TFLOP/s; None if the library is missing."""
    import ctypes as C
    path = os.path.join(ROOT, "paper_1709_00618_b200", "libtpcbench.so")
    if not os.path.exists(path):
        return None
    lib = C.CDLL(path)
    lib.tpc_bench_fp32_peak.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_void_p, C.POINTER(C.c_double)]
    out = torch.zeros(1, dtype=torch.float32, device=dev)
    tf = C.c_double(0.0)
    with torch.cuda.device(dev):
        rc = lib.tpc_bench_fp32_peak(C.c_void_p(out.data_ptr()), 4096, 5,
                                     C.c_void_p(torch.cuda.current_stream(dev).cuda_stream), C.byref(tf))
    return float(tf.value) if rc == 0 and tf.value > 0 else None


def measured_traffic(workload, windows, n_clusters):
    """dram__bytes_read.sum + dram__bytes_write.sum of the dominant kernel per launch, or None if no capture of this
    workload is committed."""
    try:
        with open(TRAFFIC_JSON) as f:
            d = json.load(f)
    except Exception:
        return None, "no committed ncu capture"
    if d.get("workload") != workload or int(d.get("windows", -1)) != int(windows) or int(d.get("n_clusters", -1)) != int(n_clusters):
        return None, f"committed capture is for {d.get('workload')} x {d.get('windows')} windows; not this workload"
    return float(d["dram_bytes_per_launch"]), f"{d['source']} (commit {d.get('commit', '?')})"


def committed_capture(workload, windows, n_clusters):
    """The other figures of the committed ncu capture (profiles/roofline_traffic.json) for this exact workload: DRAM
    bytes of the whole step and the issue statistics of the dominant kernel.  {} when the capture is of another size."""
    try:
        with open(TRAFFIC_JSON) as f:
            d = json.load(f)
    except Exception:
        return {}
    if d.get("workload") != workload or int(d.get("windows", -1)) != int(windows) or int(d.get("n_clusters", -1)) != int(n_clusters):
        return {}
    return d


def run_e2e(torch, trk, dev, layout, host_in, h_ro, batch, args, combine):
    """The whole job through tpc_pipeline_run from pinned HOST buffers: upload, tracking and download of the results
    inside the timed region (host clock around the blocking calls)."""
    from paper_1709_00618_b200.tracker import HostPipeline
    S, N = batch.n_inst, batch.n_clusters
    ipc = 36 * max(1, args.chunk_windows)
    max_chunk = max(int(batch.row_offsets[min(i + ipc, S) * batch.n_rows] - batch.row_offsets[i * batch.n_rows])
                    for i in range(0, S, ipc))
    trk.set_input_layout(layout)
    pipe = HostPipeline(trk, max_chunk, ipc, N, n_slots=args.slots, want=E2E_WANT)
    for _ in range(max(1, min(args.warmup, 2))):
        pipe.run(host_in, h_ro, S)
    torch.cuda.synchronize(dev)
    runs = []
    tw = time.perf_counter()
    for _ in range(args.steps):
        runs.append(pipe.run(host_in, h_ro, S))  # a snapshot per run (plain numbers)
    torch.cuda.synchronize(dev)
    ms = (time.perf_counter() - tw) * 1e3
    ms, n_total = combine(ms, N)
    r = runs[-1]
    k = len(runs)
    out = {"value": n_total / (ms / k * 1e-3), "unit": UNIT, "h2d_bytes_per_step": r["h2d_bytes"],
           "d2h_bytes_per_step": r["d2h_bytes"], "ms_per_step": ms / k,
           "h2d_ms": float(np.mean([x["h2d_ms"] for x in runs])),
           "compute_ms": float(np.mean([x["compute_ms"] for x in runs])),
           "d2h_ms": float(np.mean([x["d2h_ms"] for x in runs])),
           "h2d_gbs": r["h2d_bytes"] / max(np.mean([x["h2d_ms"] for x in runs]), 1e-9) / 1e6,
           "d2h_gbs": r["d2h_bytes"] / max(np.mean([x["d2h_ms"] for x in runs]), 1e-9) / 1e6,
           "chunks": r["n_chunks"], "slots": args.slots, "windows_per_chunk": args.chunk_windows,
           "gpu_launches_per_step": r["n_launches"], "tracks": r["totals"][3],
           "input": {"xyzw": "TPC_INPUT_XYZW: float4 (x, y, z, w), 16 B/cluster",
                     "yz": "TPC_INPUT_YZ: fp32 (y, z) pairs, 8 B/cluster",
                     "i16": "TPC_INPUT_I16: 16-bit fixed point (y/256 cm, z/64 cm), 4 B/cluster"}[layout],
           "results": "cluster_owner (4 B/cluster) + trk_params, trk_nhits, trk_sector per track",
           "busy": "h2d_ms / compute_ms / d2h_ms = time each stream was busy per step (CUDA events inside the "
                   "library; compute counts concurrent chunks twice); the largest one bounds the step",
           "timer": "host perf_counter around the blocking C-ABI calls"}
    pipe.close()
    trk.set_input_layout("xyzw")
    return out


def run_ours(args):
    import torch
    import torch.distributed as dist
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    skip = set(x for x in args.skip.split(",") if x)
    t_gen = time.time()
    shard = None
    if args.scaling == "strong":
        if args.windows < world:
            raise SystemExit("--scaling strong needs at least one window per rank")
        evs, batch = make_batch(args.windows, args.seed0, 0)  # the SAME job on every rank ...
        job_clusters, job_inst = batch.n_clusters, batch.n_inst
        evs, batch, shard = shard_job(evs, batch, world, rank)  # ... of which this rank tracks its block of windows
    else:
        evs, batch = make_batch(args.windows, args.seed0, rank)  # before CUDA init (fork)
    t_gen = time.time() - t_gen
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (no CPU fallback); use --impl reference for the oracle")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    from paper_1709_00618_b200 import Tracker, physics
    N, S = batch.n_clusters, batch.n_inst
    tune = json.loads(args.tune) if args.tune else {}
    trk = Tracker.for_event(batch, device=f"cuda:{local}", **tune)
    h_cl = torch.from_numpy(batch.clusters).pin_memory()
    h_ro = torch.from_numpy(batch.row_offsets).pin_memory()
    d_cl = h_cl.to(dev)
    d_ro = h_ro.to(dev)
    trk.reserve(N, S)
    trk.set_stream()
    trk.set_stage_timing(True)
    bufs, out = trk.alloc_outputs(N, trk_capacity=N // 20 + 64)
    fp32_measured = measure_fp32_peak(torch, dev)  # a few ms, before anything is timed

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize(dev)

    for _ in range(args.warmup):
        trk.track_sectors_device(d_cl, d_ro, S, out)
    barrier()
    sampler = ClockSampler(local)
    time.sleep(0.25)
    # One CUDA-event pair per step on the launching stream; the steps are queued back to back.  When the batch
    # (inputs + intermediates) could sit in the 126 MB L2, a 512 MB buffer is rewritten between steps (outside the
    # event pairs) so that every step starts cold.
    flush = (16 * N < 2 * 126e6)
    fbuf = torch.empty(512 << 20, dtype=torch.uint8, device=dev) if flush else None
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    barrier()
    t0 = time.time()
    for a, b in ev:
        if flush:
            fbuf.fill_(1)
        a.record()
        trk.track_sectors_device(d_cl, d_ro, S, out)
        b.record()
    torch.cuda.synchronize(dev)
    t1 = time.time()
    clocks = sampler.stop(t0, t1)
    ms = sum(a.elapsed_time(b) for a, b in ev)
    launches = trk.last_launch_count * args.steps
    ms, n_total = sharding.combine_step(ms, N, device=dev)  # max over ranks, total clusters (no data-path collective)
    ms_step = ms / args.steps
    value = n_total / (ms_step * 1e-3)
    # the S5 work counters (roofline arithmetic) come from one extra, untimed call of the counting variant
    trk.set_stage_timing(False)
    trk.set_work_counters(True)
    trk.track_sectors_device(d_cl, d_ro, S, out)
    torch.cuda.synchronize(dev)
    trk.set_work_counters(False)
    counts = bufs["counts"].cpu().numpy()
    all_counts = sharding.gather_counts(counts, device=dev)  # [world, 16]: job-wide totals and per-rank track bases
    # per-stage device times of the timed calls (CUDA events recorded by the library on the launching stream)
    k = min(args.steps, 32)
    st = [trk.stage_times_ms(a) for a in range(k)]  # the untimed counting call above recorded no events
    stage_ms = {nme: float(np.mean([s[nme] for s in st])) for nme in st[0]}
    own = bufs["cluster_owner"][:evs[0].n_clusters].cpu().numpy()  # window 0 of the default reading (physics report)

    # ---- the same step with the candidate lists requested (north_star: "-> candidates and fitted tracks") ------------
    with_cand = None
    if "cand" not in skip:
        cc = int(counts[1]) + 64
        d_ch = torch.empty((cc, 10), dtype=torch.int32, device=dev)
        d_cn = torch.empty(cc, dtype=torch.int32, device=dev)
        out_c = type(out).from_buffer_copy(out)  # same outputs + cand_hits / cand_n
        out_c.cand_hits, out_c.cand_n, out_c.cand_capacity = d_ch.data_ptr(), d_cn.data_ptr(), cc
        trk.set_stream()
        trk.track_sectors_device(d_cl, d_ro, S, out_c)
        evc = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(3)]
        for a, b in evc:
            a.record()
            trk.track_sectors_device(d_cl, d_ro, S, out_c)
            b.record()
        torch.cuda.synchronize(dev)
        c_ms = float(np.mean([a.elapsed_time(b) for a, b in evc]))
        with_cand = {"what": "the timed step with cand_hits / cand_n also written (the headline call passes "
                             "cand_capacity = 0: final tracks and cluster owners only)",
                     "ms_per_step": c_ms, "delta_ms": c_ms - ms_step, "value": N / (c_ms * 1e-3), "unit": UNIT,
                     "candidates": int(counts[1]), "bytes_written": int(counts[1]) * 44,
                     "cand_n_checksum": int(d_cn[:int(counts[1])].sum().item())}
        del d_ch, d_cn
        trk.track_sectors_device(d_cl, d_ro, S, out)  # phase 2 below works on the headline call's outputs
        torch.cuda.synchronize(dev)

    # ---- phase 2 on the same batch: sector merger + refit of the final tracks -----------------
    phase2 = None
    if "phase2" not in skip:
        n_trk = int(counts[3])
        p2bufs, p2o = trk.alloc_phase2(n_trk)
        evp = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(3)]
        trk.set_stream()
        trk.merge_refit_device(p2o)  # the last call on d_cl/d_ro is still the tracked one
        for a, b in evp:
            a.record()
            trk.merge_refit_device(p2o)
            b.record()
        torch.cuda.synchronize(dev)
        c2 = p2bufs["counts2"].cpu().numpy()
        p2_ms = float(np.mean([a.elapsed_time(b) for a, b in evp]))
        phase2 = {"what": "tpc_merge_refit on the final tracks of the step: refit of every track's kept hits, matching "
                          "across sector boundaries, one fit per merged track (DESIGN.md readings M1-M4)",
                  "ms": p2_ms, "tracks_in": n_trk, "merged_tracks": int(c2[0]), "links": int(c2[1]),
                  "failed_track_refits": int(c2[2]), "failed_chain_fits": int(c2[3]),
                  "gpu_launches": trk.last_launch_count, "share_of_step_plus_phase2": p2_ms / (p2_ms + ms_step)}
        del p2bufs

    # ---- end to end through the host-buffer entry point (tpc_pipeline_run) -------------------------------------------
    combine = lambda ms_, n_: sharding.combine_step(ms_, n_, device=dev)  # noqa: E731
    e2e = e2e_xyzw = e2e_yz = None
    if "e2e" not in skip:
        # the streaming configuration the library recommends: 16-bit fixed-point clusters (4 B/cluster up)
        q16, _ = datagen.quantise_i16(batch)
        h_q = torch.from_numpy(q16).pin_memory()
        e2e = run_e2e(torch, trk, dev, "i16", h_q, h_ro, batch, args, combine)
        del h_q, q16
        e2e_xyzw = run_e2e(torch, trk, dev, "xyzw", h_cl, h_ro, batch, args, combine)
        h_yz = torch.from_numpy(np.ascontiguousarray(batch.clusters[:, 1:3])).pin_memory()
        e2e_yz = run_e2e(torch, trk, dev, "yz", h_yz, h_ro, batch, args, combine)
        del h_yz

    # ---- latency of ONE drift window (CFG:4) alone on the GPU: L2 flushed before every call ----------------------
    single = None
    if "single" not in skip:
        n0, s0 = evs[0].n_clusters, evs[0].n_inst
        fb1 = fbuf if fbuf is not None else torch.empty(512 << 20, dtype=torch.uint8, device=dev)
        ev1 = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(5)]
        trk.set_stream()
        trk.track_sectors_device(d_cl[:n0], d_ro[:s0 * batch.n_rows + 1], s0, out)
        for a, b in ev1:
            fb1.fill_(1)
            a.record()
            trk.track_sectors_device(d_cl[:n0], d_ro[:s0 * batch.n_rows + 1], s0, out)
            b.record()
        torch.cuda.synchronize(dev)
        one_ms = float(np.median([a.elapsed_time(b) for a, b in ev1]))
        del fb1
        single = {"workload": "cfg4: one drift window alone (36 sector instances), L2 flushed", "ms": one_ms,
                  "clusters": n0, "clusters_per_s": n0 / (one_ms * 1e-3)}

    # ---- the same batch with S2 row bridging on (reading A2'; not the headline reading) ------
    bridge = None
    if "bridge" not in skip:
        trk_b = Tracker.for_event(batch, device=f"cuda:{local}", **{**tune, "nf_bridge_rows": 1})
        trk_b.reserve(N, S)
        trk_b.set_stream()
        trk_b.set_stage_timing(True)
        for _ in range(2):
            trk_b.track_sectors_device(d_cl, d_ro, S, out)
        evb = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(3)]
        for a, b in evb:
            a.record()
            trk_b.track_sectors_device(d_cl, d_ro, S, out)
            b.record()
        torch.cuda.synchronize(dev)
        bridge_ms = float(np.mean([a.elapsed_time(b) for a, b in evb]))
        cb = bufs["counts"].cpu().numpy()
        stb = [trk_b.stage_times_ms(a) for a in range(3)]
        own_b = bufs["cluster_owner"][:evs[0].n_clusters].cpu().numpy()
        bridge = {"reading": "nf_bridge_rows=1: a hit without an admissible adjacent pair may take one partner two "
                             "rows away (DESIGN.md A2'); parity-tested against the oracle like the default reading",
                  "value": N / (bridge_ms * 1e-3), "unit": UNIT, "ms_per_step": bridge_ms,
                  "stage_ms": {nme: float(np.mean([x[nme] for x in stb])) for nme in stb[0]},
                  "results": {"candidates": int(cb[1]), "tracklets": int(cb[2]), "tracks": int(cb[3]),
                              "track_hits": int(cb[4])},
                  "physics_window0": physics.report(evs[0], own_b, int(own_b.max()) + 1 if (own_b >= 0).any() else 0)}
        trk_b.close()

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return
    hbm_peak, sm_max, peak_src = measured_peaks()
    fp32_peak = N_SM * FP32_LANES_PER_SM * 2 * sm_max * 1e6 / 1e12  # TFLOP/s
    # follow_kernel alone: the work of the fit kernel (the candidates' own hits, counts[11..12]) is not its work
    tr_f, up_f = int(counts[6] - counts[11]), int(counts[7] - counts[12])
    flops = (tr_f * FLOP_TRANSPORT + up_f * FLOP_UPDATE + counts[8] * FLOP_EXAMINE + counts[9] * FLOP_SEARCH)
    t_follow = stage_ms["follow"] * 1e-3
    ach = flops / t_follow / 1e12
    traffic, traffic_src = measured_traffic(WORKLOAD, args.windows, N)
    roof = {"kernel": "follow_kernel (S5 Kalman track following, row-by-row extrapolation)", "bound": "alu",
            "achieved": ach, "peak": fp32_peak, "unit": "TFLOP/s", "frac": ach / fp32_peak,
            "traffic": traffic, "traffic_source": traffic_src,
            "peak_source": f"NOMINAL, not measured: 148 SM x 128 fp32 lanes x 2 flop x {sm_max:.0f} MHz (DESIGN.md); "
                           "MEASURED_PEAKS.json holds no fp32 ALU figure",
            "avg_launch_ms": stage_ms["follow"], "share_of_step": stage_ms["follow"] / sum(stage_ms.values()),
            "algorithmic_flop_per_launch": float(flops),
            "work": {"transports": tr_f, "updates": up_f, "clusters_examined": int(counts[8]),
                     "searches": int(counts[9]), "fit_kernel_transports": int(counts[11]),
                     "fit_kernel_updates": int(counts[12]), "row_steps_per_cluster": float(counts[6]) / N},
            "hbm_view": {"bytes_per_cluster": BYTES_PER_CLUSTER_S5,
                         "achieved_gbs": BYTES_PER_CLUSTER_S5 * N / t_follow / 1e9,
                         "frac_of_hbm_peak": BYTES_PER_CLUSTER_S5 * N / t_follow / 1e9 / hbm_peak}}
    path_gbs = BYTES_PER_CLUSTER_PATH * N / (ms_step * 1e-3) / 1e9
    roof_path = {"bound": "hbm", "achieved": path_gbs, "peak": hbm_peak, "unit": "GB/s", "frac": path_gbs / hbm_peak,
                 "bytes_per_cluster_model": BYTES_PER_CLUSTER_PATH, "peak_source": peak_src,
                 "frac_of_nominal_8TBs": path_gbs / 8000.0}
    if fp32_measured:
        roof["peak_measured"] = {"value": fp32_measured, "unit": "TFLOP/s", "frac": ach / fp32_measured,
                                 "frac_of_nominal": fp32_measured / fp32_peak,
                                 "how": "FMA chains (8 per thread, 64 warps per SM), best of 5 launches, CUDA events; "
                                        "paper_1709_00618_b200/csrc_bench/fp32_peak.cu, run at the start of this bench"}
    # SURVEY 8(d)'s headline fraction and the issue view of the dominant kernel go INSIDE `roofline` (the key the
    # driver's record keeps); `roofline_path_hbm` stays as before for readers of earlier rounds' lines.
    cap = committed_capture(WORKLOAD, args.windows, N)
    roof["path_hbm"] = dict(roof_path)
    if cap.get("step_dram_bytes"):
        nb = float(cap["step_dram_bytes"])
        roof["path_hbm"].update({
            "ncu_dram_bytes_per_step": nb, "ncu_bytes_per_cluster": nb / N,
            "ncu_over_model": nb / (BYTES_PER_CLUSTER_PATH * N),
            "dram_gbs_at_ncu_bytes": nb / (ms_step * 1e-3) / 1e9,
            "ncu_source": cap.get("step_dram_source", ""),
            "rule": "SURVEY 8(d): achieved = min(ncu bytes, model bytes per cluster x N) / step time"})
    if cap.get("warp_instructions_per_launch"):
        wi = float(cap["warp_instructions_per_launch"])
        slots = N_SM * 4 * sm_max * 1e6 * t_follow  # 4 schedulers per SM, one warp instruction per cycle each
        roof["issue"] = {"warp_instructions_per_launch": wi, "issue_slots_per_launch": slots,
                         "frac_of_issue_slots": wi / slots, "ncu_issue_active": cap.get("issue_active"),
                         "lanes_per_instruction": cap.get("lanes_per_instruction"),
                         "lane_instructions_per_row_step": wi * float(cap.get("lanes_per_instruction", 32.0)) / max(tr_f, 1),
                         "source": f"{cap.get('issue_source', '')} (commit {cap.get('commit', '?')}); the slot count "
                                   "uses this run's measured launch time"}
    if e2e is not None:
        def _sub(x):
            return None if x is None else {k: x[k] for k in ("value", "unit", "ms_per_step", "h2d_bytes_per_step",
                                                             "d2h_bytes_per_step", "h2d_ms", "compute_ms", "d2h_ms",
                                                             "input")}
        e2e["fp32_yz"] = _sub(e2e_yz)
        e2e["fp32_xyzw"] = _sub(e2e_xyzw)
        e2e["series_note"] = ("the headline e2e streams the 16-bit fixed-point layout (SURVEY 8(f) NEXT-4, "
                              "parity-tested against the oracle on the decoded coordinates) and downloads "
                              "cluster_owner + trk_params/trk_nhits/trk_sector; BASELINE.json configs[4] names fp32 "
                              "clusters: that figure is fp32_yz (same tracker results as float4, bit for bit) and "
                              "fp32_xyzw (the round-1 layout).  Round 1's e2e uploaded float4 and downloaded all seven "
                              "result arrays incl. trk_cov and trk_hits, so the series breaks between rounds 1 and 2")
    cpu = None
    if world == 1 and "cpu" not in skip:
        cpu, _ = cpu_baseline(evs, 1)
    n_trk0 = int(own.max()) + 1 if (own >= 0).any() else 0
    phys = physics.report(evs[0], own, n_trk0)
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_step, "higher_is_better": True, "scaling": args.scaling,
            "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": f"{'cfg5 throughput batch' if WORKLOAD == 'cfg5' else WORKLOAD + ' batch'}: "
                                   f"{args.windows} {WORKLOADS[WORKLOAD]} per GPU in one call",
                       "windows_per_gpu": args.windows, "sector_instances_per_gpu": S, "clusters_per_gpu": N,
                       "ms_per_window": ms_step / args.windows, "seed0": args.seed0,
                       "l2": (f"inputs are {16 * N / 1e6:.0f} MB of float4; " +
                              ("L2 flushed (512 MB write) before every timed step" if flush else
                               "larger than twice the 126 MB L2, steps run back to back without a flush")),
                       "generation_s": round(t_gen, 1)},
            "clocks": clocks, "gpu_launches": launches,
            "e2e": e2e, "e2e_xyzw_f32": e2e_xyzw, "e2e_yz_f32": e2e_yz,
            "roofline": roof, "roofline_path_hbm": roof_path, "cpu_baseline": cpu,
            "stage_ms": stage_ms, "with_candidates": with_cand, "phase2_merge_refit": phase2, "single_window": single,
            "results": {"candidates": int(counts[1]), "tracklets": int(counts[2]), "tracks": int(counts[3]),
                        "track_hits": int(counts[4]), "error_flags": int(counts[5])},
            "physics_window0": phys,
            "next1_bridge_rows": bridge}
    if world > 1 or shard is not None:
        line["all_ranks"] = {"tracks": int(all_counts[:, 3].sum()), "candidates": int(all_counts[:, 1].sum()),
                             "track_base_per_rank": [int(x) for x in np.concatenate([[0], np.cumsum(all_counts[:-1, 3])])]}
    if shard is not None:
        line["config"]["strong_scaling_job"] = {
            "what": "ONE job of --windows drift windows for all ranks; contiguous blocks of whole windows per rank, "
                    "balanced by cluster count (sharding.partition_instances); no data-path collective",
            "job_clusters": job_clusters, "job_sector_instances": job_inst, "rank0_shard": shard}
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--windows", type=int, default=100, help="CFG:4 drift windows per GPU and step")
    ap.add_argument("--chunk-windows", type=int, default=10, help="windows per upload chunk in the e2e pipeline")
    ap.add_argument("--slots", type=int, default=3)
    ap.add_argument("--workload", default="cfg5", choices=sorted(WORKLOADS),
                    help="what --windows counts: drift windows (default, the headline), or CFG:3 / CFG:2 events for the "
                         "linear-scaling check of PAPER.md:33")
    ap.add_argument("--scaling", default="weak", choices=["weak", "strong"],
                    help="weak (default, what the driver runs): every rank tracks its own --windows windows; strong: "
                         "ONE job of --windows windows is partitioned over the ranks (SURVEY 8(e))")
    ap.add_argument("--seed0", type=int, default=5001)
    ap.add_argument("--tune", default="", help='JSON dict of performance-only tracker parameters, e.g. {"grid_cells_y": 8}')
    ap.add_argument("--skip", default="", help="comma list of optional sections to leave out: e2e,phase2,single,bridge,cpu,cand")
    args = ap.parse_args()
    global WORKLOAD
    WORKLOAD = args.workload
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
