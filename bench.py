#!/usr/bin/env python
"""bench.py -- TPC time-frame tracking throughput on B200 (metric of BASELINE.json: clusters tracked per second,
ms per 10 ms time frame, HBM GB/s vs peak).

A "step" is one pass of the whole hot path (C1 ingest -> C2 finder -> C3/C4 cleaner + start hits -> C5 tracklet
constructor -> C6 selector) over one synthetic continuous-readout time frame (configs[3] of BASELINE.json: 10 ms at
50 kHz, ~500 collisions).  `value` is measured with the clusters resident in HBM; `e2e` goes through the C-ABI host
entry point with pinned HOST buffers (H2D of the clusters and D2H of the tracks inside the timed region).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config 3] [--frame-us F] [--impl reference]

N > 1 (torchrun, one rank per GPU): every rank tracks its own time frame (the paper's farm runs independent time
frames per GPU) -> weak scaling, no data-path collective.  `--shard sectors` instead cuts ONE frame by sector
across the ranks (strong scaling, still no collective inside the tracking; paper_2102_08862_b200/shard.py).
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

CONFIG_NAMES = {0: "configs[0] single sector, 300 tracks", 1: "configs[1] full TPC, one 4000-track collision",
                2: "configs[2] 2 ms continuous readout at 50 kHz", 3: "configs[3] 10 ms continuous readout at 50 kHz",
                4: "configs[4] 10 ms high-occupancy stress frame"}

# Algorithmic HBM bytes per cluster of each step: SURVEY.md §8(d)'s per-unit figures (what the METHOD must move, whatever
# sort or layout this implementation uses).  ingest: 12 read + 12 read again + 12 write (+ 4 grid) = 40, split
# over its two kernels; finder 24; cleaner + start hits 24, split over its two steps; tracklet_init: seeds + chain walk
# (32 B + 6.8 chain hits x 16 B per tracklet, 0.076 tracklets per cluster) = 11; selector 60 = claim 30 + count 26 + emit 4.
ALGO_BYTES_PER_CLUSTER = {
    "ingest_radix_sort": 36, "grid_build": 4,
    "neighbours_finder": 24, "cleaner_start_hits": 20, "start_hit_compaction": 4, "tracklet_init": 11,
    "selector_claim": 30, "selector_count": 26, "selector_scan": 0, "selector_emit": 4,
}
# Tracklet constructor: bound by plain fp32 ALU issue.  Algorithmic lane-instructions of one row step
# (= one transport [+ search] [+ update]) counted from the statement lists of DESIGN.md §3 with IEEE division and
# square root ~ 8 instructions each: transport 123, update 52 x 0.85 of steps, search 12 per candidate.
ALGO_LANE_INST_TRANSPORT, ALGO_LANE_INST_UPDATE, ALGO_LANE_INST_PER_CANDIDATE = 123, 52, 12
TRACKLET_PHASES = {"tracklet_fit_up": "fit_up", "tracklet_follow_up": "follow_up", "tracklet_fit_down": "fit_down",
                   "tracklet_follow_down": "follow_down"}     # step name -> work-counter group
# roofline.traffic: dram__bytes_read.sum + dram__bytes_write.sum per launch, read from the committed summary of the
# `ncu --set full` capture of configs[3], seed 1 (profiles/NCU_TRAFFIC_CSV; its .md names the command and the commit it was
# taken at).  Reported for that workload only, null otherwise.
NCU_TRAFFIC_CSV = "r02_ncu_traffic_config3.csv"
STEP_KERNEL = {"tracklet_follow_up": "k_tracklet_follow<0>", "tracklet_follow_down": "k_tracklet_follow<1>",
               "tracklet_fit_up": "k_tracklet_fit<0>", "tracklet_fit_down": "k_tracklet_fit<1>", "neighbours_finder": "k_neighbours_finder",
               "selector_claim": ("k_selector_claim_top", "k_selector_claim"), "selector_count": "k_selector_count_hits",
               "tracklet_init": "k_tracklet_init"}       # a step of several kernels: their traffic is summed


def _ncu_traffic():
    """{kernel name: (bytes per launch, commit)} from profiles/NCU_TRAFFIC_CSV; {} if the file is missing."""
    out = {}
    try:
        with open(os.path.join(ROOT, "profiles", NCU_TRAFFIC_CSV)) as f:
            for line in f:
                q = [x.strip() for x in line.split(",")]
                if len(q) >= 4 and q[0] != "kernel" and not q[0].startswith("#"):
                    out[q[0]] = (float(q[1]) + float(q[2]), q[3])
    except OSError:
        pass
    return out
def _cpu_model():
    try:
        with open("/proc/cpuinfo") as f:
            for line in f:
                if line.startswith("model name"):
                    return line.split(":", 1)[1].strip()
    except OSError:
        pass
    return None


def _step_traffic(traffic, step):
    """(bytes per launch summed over the step's kernels, commit) or None."""
    ks = STEP_KERNEL.get(step, ())
    ks = (ks,) if isinstance(ks, str) else ks
    got = [traffic[k] for k in ks if k in traffic]
    return (sum(g[0] for g in got), got[0][1]) if got and len(got) == len(ks) else None


SM_COUNT, SMSP_PER_SM, LANES = 148, 4, 32      # B300_MICROARCH.md: 4 schedulers per SM, <= 1 warp instruction per cycle each


def _peaks():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            p = json.load(f)
        return float(p["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """Samples SM clock and throttle reasons with nvidia-smi during the timed region."""

    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.samples, self._stop, self._th = index, [], threading.Event(), None

    def _run(self):
        while not self._stop.is_set():
            try:
                out = subprocess.run(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits"],
                                     capture_output=True, text=True, timeout=5).stdout.strip()
                if out:
                    self.samples.append([x.strip() for x in out.split(",")])
            except Exception:
                pass
            self._stop.wait(0.1)

    def __enter__(self):
        self._th = threading.Thread(target=self._run, daemon=True)
        self._th.start()
        return self

    def __exit__(self, *a):
        self._stop.set()
        self._th.join(timeout=6)

    def summary(self):
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for s in self.samples:
            try:
                sm.append(float(s[0])); mx.append(float(s[1]))
                for nm, v in zip(names, s[3:7]):
                    if v.lower().startswith("active"):
                        reasons.add(nm)
            except Exception:
                continue
        sm.sort()
        return {"sm_mhz": (sm[len(sm) // 2] if sm else None), "sm_max_mhz": (max(mx) if mx else None),
                "reasons": sorted(reasons), "samples": len(sm)}


def _tracker_params(T, cfg, n, host_staging, profile, grid=(0, 0, 0), follower=0):
    p = T.default_params(cfg.sigma_y_cm, cfg.sigma_z_cm, max_clusters=n)
    p.follower = int(follower)
    p.host_staging, p.profile, p.grid_time_bins, p.grid_pad_bins = int(host_staging), int(profile), int(grid[0]), int(grid[1])
    p.slice_time_bins = int(grid[2])
    return p


def _cpu_oracle_run(cid, seed, frame_us):
    """Times the oracle, as it stands, on one host core over a bounded sample of the workload."""
    import oracle
    from paper_2102_08862_b200 import gen
    cfg = gen.preset(cid, seed, frame_us if cid >= 2 else None)
    tf = gen.generate(cfg, want_truth=False)
    g = oracle.default_geometry(cfg.n_sectors, tf.max_time_bin)
    p = oracle.default_params(cfg.sigma_y_cm, cfg.sigma_z_cm)
    t0 = time.perf_counter()
    r = oracle.track(g, p, tf.row, tf.pad, tf.time)
    dt = time.perf_counter() - t0
    return tf.n, dt, len(r.tr_seed)


def _cpu_oracle_run_all_cores(cid, seed, frame_us, tf=None):
    """The same unchanged oracle, one call per sector (sectors are independent), from a thread pool: BASELINE.md §3 (2).
    ctypes releases the GIL during the call.  Returns (clusters, seconds, threads used, tracks).  `tf`: a frame that is
    already generated (the WHOLE benchmark frame); else the generator's frame cut to frame_us."""
    import numpy as np
    from concurrent.futures import ThreadPoolExecutor
    import oracle
    from paper_2102_08862_b200 import gen
    cfg = gen.preset(cid, seed, frame_us if cid >= 2 else None)
    if tf is None:
        tf = gen.generate(cfg, want_truth=False)
    n_rows = 152
    sec = (tf.row.astype(np.int64) // n_rows)
    parts = []
    for s_ in range(cfg.n_sectors):                      # split outside the timed region (the input of a per-sector tracker)
        m = np.nonzero(sec == s_)[0]
        parts.append((np.ascontiguousarray(tf.row[m] - np.float32(s_ * n_rows)), np.ascontiguousarray(tf.pad[m]),
                      np.ascontiguousarray(tf.time[m])))
    g1 = oracle.default_geometry(1, tf.max_time_bin)
    p = oracle.default_params(cfg.sigma_y_cm, cfg.sigma_z_cm)
    threads = max(1, min(len(parts), os.cpu_count() or 1))
    oracle.lib()
    t0 = time.perf_counter()
    with ThreadPoolExecutor(threads) as ex:
        res = list(ex.map(lambda a: len(oracle.track(g1, p, *a).tr_seed), parts))
    dt = time.perf_counter() - t0
    return tf.n, dt, threads, int(sum(res))


def run_reference(args):
    """--impl reference: the CPU oracle, as it stands, on the box's host cores (one unchanged call per sector from a thread
    pool: sectors are independent), same metric; each step a bounded sample of the workload (the frame cut to
    --ref-frame-us) so that the whole run ends within a few minutes."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    cid = args.config
    sample_us = args.ref_frame_us
    total_n, total_t, cores = 0, 0.0, 1
    for i in range(args.warmup + args.steps):
        if cid >= 1:
            n, dt, cores, _ = _cpu_oracle_run_all_cores(cid, 1000 + i, sample_us)
        else:
            n, dt, _ = _cpu_oracle_run(cid, 1000 + i, sample_us)
        if i >= args.warmup:
            total_n += n; total_t += dt
    value = total_n / total_t
    sample = (f"{CONFIG_NAMES[cid]} generator with the frame cut to {sample_us:g} us per step"
              if cid >= 2 else CONFIG_NAMES[cid])
    line = {"impl": "reference", "metric": "tpc_clusters_tracked_per_s", "value": value, "unit": "clusters/s",
            "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * total_t / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": CONFIG_NAMES[cid], "sample": sample, "clusters_per_step": total_n // args.steps},
            "cpu_baseline": {"value": value, "unit": "clusters/s", "cores": cores, "kind": "oracle", "sample": sample, "cpu_model": _cpu_model()},
            "e2e": {"value": value, "unit": "clusters/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=3, help="BASELINE.json configs index (default 3: the 10 ms frame)")
    ap.add_argument("--frame-us", type=float, default=None, help="override the frame length (smoke runs only)")
    ap.add_argument("--seed", type=int, default=1)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--ref-frame-us", type=float, default=1000.0, help="frame length of one reference-arm step")
    ap.add_argument("--cpu-sample-us", type=float, default=150.0, help="frame length of the single-core cpu_baseline sample")
    ap.add_argument("--cpu-whole-frame", type=int, default=1, help="1: time the all-cores oracle on the WHOLE benchmark frame (about 20 s)")
    ap.add_argument("--grid-time-bins", type=int, default=0, help="grid bin width in time bins (0 = library default)")
    ap.add_argument("--slice-time-bins", type=int, default=0, help="processing-order time slice (0 = library default)")
    ap.add_argument("--grid-pad-bins", type=int, default=0, help="grid bins across a pad row (0 = library default)")
    ap.add_argument("--shard", default="frames", choices=["frames", "sectors"],
                    help="N > 1: frames = every rank tracks its own frame (replicas, weak scaling; the default); sectors = ONE frame cut by "
                         "sector across the ranks (strong scaling; paper_2102_08862_b200/shard.py)")
    ap.add_argument("--shard-of", default="", help="W:R with --shard sectors in a single process: track the sectors rank R of W ranks would get "
                                                  "(the per-rank work of a W-GPU job measured on one GPU; value then covers that shard only)")
    ap.add_argument("--follower", type=int, default=0, help="0 = per-lane follower (default), 1 = row-synchronous follower (A/B)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-cluster-finder", action="store_true")
    ap.add_argument("--cf-frame-us", type=float, default=1000.0, help="frame length whose samples the cluster finder (C0) is timed on")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--e2e-inflight", type=int, default=3, help="time frames in flight in the end-to-end measurement (measured: 1: 110.6 ms, 2: 75.6, 3: 71.5, 4: 73.5 per frame)")
    args = ap.parse_args()
    if args.warmup < 3:
        args.warmup = 3
    if args.impl == "reference":
        return run_reference(args)

    import numpy as np
    import torch
    import torch.distributed as dist
    from paper_2102_08862_b200 import gen, replicas, tracker as T

    rank, world, local_rank = replicas.rank_world_local()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the tracker has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    # ---- synthetic time frame (one per rank; seeded) ----
    cid = args.config
    by_sector = args.shard == "sectors"
    cfg = gen.preset(cid, args.seed if by_sector else replicas.frame_seed(args.seed, rank), args.frame_us if cid >= 2 else None)
    cfg.n_threads = max(1, (os.cpu_count() or 8) // max(world, 1))
    t_gen = time.perf_counter()
    tf = gen.generate(cfg, want_truth=False)
    t_gen = time.perf_counter() - t_gen
    sector_range = None
    if by_sector:                                    # every rank holds the same frame and keeps the clusters of its sectors, in order
        import dataclasses
        from paper_2102_08862_b200 import shard
        n_rows = 152
        w_eff, r_eff = (int(v) for v in args.shard_of.split(":")) if (args.shard_of and world == 1) else (world, rank)
        sector_range = shard.sector_ranges(cfg.n_sectors, w_eff, shard.sector_histogram(tf.row, cfg.n_sectors, n_rows))[r_eff]
        sel = shard.shard_indices(tf.row, n_rows, *sector_range)
        tf = dataclasses.replace(tf, row=np.ascontiguousarray(tf.row[sel]), pad=np.ascontiguousarray(tf.pad[sel]),
                                 time=np.ascontiguousarray(tf.time[sel]), charge=np.ascontiguousarray(tf.charge[sel]),
                                 truth_track=tf.truth_track[:0], truth_arc=tf.truth_arc[:0])
    n = tf.n
    host = [torch.from_numpy(a).pin_memory() for a in (tf.row, tf.pad, tf.time)]
    devc = [h.to(dev, non_blocking=True) for h in host]
    torch.cuda.synchronize()

    g = T.default_geometry(cfg.n_sectors, tf.max_time_bin)
    gp = (args.grid_time_bins, args.grid_pad_bins, args.slice_time_bins)
    trk = T.Tracker(g, _tracker_params(T, cfg, n, False, False, gp, args.follower), device=str(dev))     # `value`: no per-step events
    outs = trk.alloc_outputs(n)
    stream = torch.cuda.Stream(device=dev)

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident timing ----
    with torch.cuda.stream(stream):
        for _ in range(args.warmup):
            trk.tpc_track_timeframe(*devc, n=n, outputs=outs, stream=stream)
    barrier()
    step_acc = {}
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    with ClockSampler(local_rank) as clocks:
        barrier()
        with torch.cuda.stream(stream):
            e0.record(stream)
            for _ in range(args.steps):
                trk.tpc_track_timeframe(*devc, n=n, outputs=outs, stream=stream)
            e1.record(stream)
        barrier()
    total_ms = e0.elapsed_time(e1)
    launches = trk.last_launches() * args.steps
    # the same call captured once in a CUDA graph and replayed (the call only enqueues work, so it can be captured): what a
    # caller gains on frames whose launches cost more than their kernels (configs[0], [1]); not part of `value`
    graph_replay = None
    try:
        gr = torch.cuda.CUDAGraph()
        torch.cuda.synchronize()
        with torch.cuda.graph(gr, stream=stream):
            trk.tpc_track_timeframe(*devc, n=n, outputs=outs, stream=torch.cuda.current_stream(dev))
        with torch.cuda.stream(stream):
            for _ in range(args.warmup):
                gr.replay()
            g0, g1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            g0.record(stream)
            for _ in range(args.steps):
                gr.replay()
            g1.record(stream)
        stream.synchronize()
        graph_replay = {"ms_per_step": g0.elapsed_time(g1) / args.steps, "eager_ms_per_step_this_rank": total_ms / args.steps,
                        "kernels_per_graph": trk.last_launches()}
        del gr
    except Exception as e:                            # reported, never fatal: the eager numbers above stand
        graph_replay = {"error": repr(e)[:200]}
    trk.close()
    del trk
    # per-kernel durations: CUDA events recorded by the library on the same stream (a second handle with
    # params.profile = 1), averaged over a few extra steps
    trk = T.Tracker(g, _tracker_params(T, cfg, n, False, True, gp, args.follower), device=str(dev))
    n_prof = min(args.steps, 5)
    for _ in range(n_prof):
        with torch.cuda.stream(stream):
            trk.tpc_track_timeframe(*devc, n=n, outputs=outs, stream=stream)
        stream.synchronize()
        for k, v in trk.step_ms().items():
            step_acc[k] = step_acc.get(k, 0.0) + v / n_prof
    work = trk.work_counters(stream)
    n_tracks = int(outs[0].n_tracks[0])
    n_track_hits = int(outs[0].n_track_hits[0])
    status = int(outs[0].status[0])
    arena_gb = trk.arena_bytes / 1e9
    alu_measured = T.tpc_selftest_alu_peak(stream)       # (scalar fp32 lane-inst/s, packed f32x2 fp32 ops/s), this GPU, now
    # ---- widening step C7 (sector-boundary merging of the tracks, not part of `value`): timed on its own ----
    merge = None
    if cfg.n_sectors >= 18:
        m0, m1, m2, m3, m4, m5, m6 = (torch.cuda.Event(enable_timing=True) for _ in range(7))
        merged = refit = ce = comp = full = full_ce = None
        ms_m = ms_r = ms_c = ms_q = ms_f = ms_fc = 0.0
        outs_c = trk.alloc_outputs(n, hit_coords=True)      # C8 reads the hits' coordinates from two optional emit outputs
        for _ in range(3):
            with torch.cuda.stream(stream):
                trk.tpc_track_timeframe(*devc, n=n, outputs=outs_c, stream=stream)    # the merger's input (and it reuses the arena)
                m0.record(stream)
                merged = trk.tpc_merge_tracks(outs_c, merged=merged, stream=stream)
                m1.record(stream)
                refit = trk.tpc_refit_chains(outs_c, merged, refit=refit, stream=stream)
                m2.record(stream)
                ce = trk.tpc_merge_central_electrode(outs_c, merged=ce, stream=stream)
                m3.record(stream)
                comp = trk.tpc_compress_tracks(outs_c, n, out=comp, stream=stream)
                m4.record(stream)
                full = trk.tpc_refit_full(outs_c, merged, out=full, stream=stream)
                m5.record(stream)
                full_ce = trk.tpc_refit_full(outs_c, merged, out=full_ce, stream=stream, ce_merged=ce)
                m6.record(stream)
            stream.synchronize()
            ms_m, ms_r, ms_c, ms_q, ms_f, ms_fc = (m0.elapsed_time(m1), m1.elapsed_time(m2), m2.elapsed_time(m3), m3.elapsed_time(m4),
                                                   m4.elapsed_time(m5), m5.elapsed_time(m6))      # last of three
        emit_with_coords_ms = trk.step_ms().get("selector_emit")
        merge = {"step": "sector_boundary_merge (C7, tpc_merge_tracks)", "ms": round(ms_m, 4), "n_links": int(merged[3][0]),
                 "n_tracks": n_tracks, "tracks_per_s": n_tracks / (ms_m * 1e-3) if ms_m > 0 else None,
                 "gpu_launches": 8, "in_value": False,
                 "refit": {"step": "chain_refit (C8, tpc_refit_chains)", "ms": round(ms_r, 4), "n_chains_refitted": int((refit[0] == 1).sum()),
                           "n_chains_failed": int((refit[0] == -1).sum()), "hits_refitted": int(refit[1][refit[0] == 1].sum()),
                           "gpu_launches": trk.last_merge_launches(),
                           "selector_emit_ms_with_hit_coordinates": emit_with_coords_ms},
                 "central_electrode": {"step": "central_electrode_merge (C10, tpc_merge_central_electrode)", "ms": round(ms_c, 4),
                                       "n_links": int(ce[3][0]), "gpu_launches": 7}}
        # C12: every chain root refitted with the full 5x5 covariance and the material of the gas.  ALU-bound like C5: 371 lane-
        # instructions per hit with §6's convention (division, square root = 8): step 179 + 5 div + 5 sqrt = 259, two scalar
        # updates 94 + 2 div = 110, measurement 2
        hits_full = int(full[1][full[0] == 1].sum())
        merge["full_refit"] = {"step": "full_covariance_refit (C12, tpc_refit_full)", "ms": round(ms_f, 4),
                               "n_roots_refitted": int((full[0] == 1).sum()), "n_roots_failed": int((full[0] == -1).sum()),
                               "hits_refitted": hits_full, "hits_per_s": hits_full / (ms_f * 1e-3) if ms_f > 0 else None,
                               "bound": "alu", "lane_inst_per_hit": 371,
                               "achieved_T_lane_inst_per_s": round(371 * hits_full / (ms_f * 1e-3) / 1e12, 3) if ms_f > 0 else None,
                               "gpu_launches": 2,
                               "across_the_central_electrode": {"step": "tpc_refit_full_ce (C12 over C7 + C10 links)", "ms": round(ms_fc, 4),
                                                                "n_roots_refitted": int((full_ce[0] == 1).sum()),
                                                                "n_chains_through_the_electrode": int(((full_ce[1] > full[1]) & (full_ce[0] == 1)).sum())}}
        # C11: hit rejection + track-model residual symbols; their entropy (a host-side measurement of the output, numpy)
        # beside the entropy of the same hits' raw coordinates at the same quantisation
        ok_c = comp[1][:n_tracks].cpu().numpy()
        nh_c = outs_c[0].n_hits[:n_tracks].cpu().numpy()
        coded = np.repeat(ok_c == 1, nh_c)
        def _entropy(x):
            c = np.bincount((x.astype(np.int64) - int(x.min())))
            pr = c[c > 0] / x.size
            return float(-(pr * np.log2(pr)).sum())
        qy_c, qz_c = comp[2][:n_track_hits].cpu().numpy()[coded], comp[3][:n_track_hits].cpu().numpy()[coded]
        hi_c = outs_c[0].hit_index[:n_track_hits].cpu().numpy()[coded]
        raw_bits = _entropy(np.rint(tf.pad[hi_c].astype(np.float64) * 0.5 / 0.025).astype(np.int64)) + \
            _entropy(np.rint(tf.time[hi_c].astype(np.float64) * 0.516 / 0.025).astype(np.int64))
        merge["compression"] = {"step": "hit_rejection + residual_coding (C11, tpc_compress_tracks)", "ms": round(ms_q, 4),
                                "hits_coded": int(coded.sum()), "hits_coded_per_s": float(coded.sum()) / (ms_q * 1e-3),
                                "tracks_rejected": int((ok_c == -1).sum()), "tracks_not_coded": int((ok_c == 0).sum()),
                                "hits_rejected": int(comp[0][:n].sum().item()), "step_cm": 0.025,
                                "entropy_bits_per_hit_symbols": round(_entropy(qy_c) + _entropy(qz_c), 3),
                                "entropy_bits_per_hit_raw_coordinates_same_step": round(raw_bits, 3), "gpu_launches": 2}
        del outs_c
    # ---- widening step C0 (the cluster finder in front of the path, not part of `value`): timed on the samples of a 1 ms
    # cut of the same generator (digitising the whole 10 ms frame would be 9e8 samples / 14 GB of host work per run)
    cluster_finder = None
    if not args.no_cluster_finder:
        ccfg = gen.preset(cid, args.seed, min(args.cf_frame_us, cfg.frame_us) if cid >= 2 else None)
        ccfg.n_threads = cfg.n_threads
        ctf = gen.generate(ccfg, want_truth=False)
        dg = gen.digitize(ctf.row, ctf.pad, ctf.time, ctf.charge, ccfg.n_sectors, ctf.max_time_bin)
        dd = [torch.from_numpy(a).to(dev) for a in (dg.row, dg.pad, dg.time, dg.adc)]
        cf_out = None
        c0, c1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        n_rep = 5
        for i in range(3 + n_rep):
            if i == 3:
                c0.record(stream)
            with torch.cuda.stream(stream):
                cf_out = trk.tpc_find_clusters(*dd, n=dg.n, out=cf_out, stream=stream)
        c1.record(stream)
        stream.synchronize()
        ms_cf = c0.elapsed_time(c1) / n_rep
        k_cf = int(cf_out[4][0])
        cf_bytes = 16 * dg.n + 16 * k_cf
        cluster_finder = {"step": "cluster_finder (C0, tpc_find_clusters)", "ms": round(ms_cf, 4), "n_samples": dg.n, "n_clusters": k_cf,
                          "samples_per_s": dg.n / (ms_cf * 1e-3), "clusters_per_s": k_cf / (ms_cf * 1e-3),
                          "sample": f"samples of the same generator cut to {ccfg.frame_us:g} us ({ctf.n} generated clusters)" if cid >= 2 else "the whole frame",
                          "bound": "hbm", "achieved": round(cf_bytes / (ms_cf * 1e-3) / 1e9, 1), "unit": "GB/s",
                          "algo_bytes": "16 per sample read + 16 per cluster written", "gpu_launches": trk.last_merge_launches(), "in_value": False}
        if not args.no_cpu_baseline and rank == 0:          # the C0 oracle beside it, one core, on the first 3e6 samples
            from oracle import clusterfinder as CFO
            m = min(dg.n, 3_000_000)
            t0 = time.perf_counter()
            CFO.find_clusters(dg.row[:m], dg.pad[:m], dg.time[:m], dg.adc[:m])
            dt = time.perf_counter() - t0
            cluster_finder["cpu_baseline"] = {"value": m / dt, "unit": "samples/s", "cores": 1, "kind": "oracle", "sample": f"the first {m} samples", "seconds": dt}
        del dd, cf_out
    trk.close()
    del trk, outs

    # whole-job numbers: time = max over ranks, work = sum over ranks (paper_2102_08862_b200/replicas.py)
    ms_per_step, value, n_all = replicas.aggregate(total_ms, n, args.steps, world, device=dev)

    # ---- end to end through the C-ABI host entry point (pinned host buffers) ----
    # Every step copies the frame host->device, tracks it and copies the tracks back, all inside tpc_track_timeframe_host.
    # `--e2e-inflight 3` (default) keeps three frames in flight on three handles / streams / host threads, the way a
    # processing node buffers time frames: the PCIe copies of one frame overlap the kernels of another.
    e2e = None
    if not args.no_e2e:
        def measure_e2e(n_fl):
            trks = [T.Tracker(g, _tracker_params(T, cfg, n, True, False, gp, args.follower), device=str(dev)) for _ in range(n_fl)]
            houts = [t.alloc_outputs(n, host=True) for t in trks]
            streams = [torch.cuda.Stream(device=dev) for _ in range(n_fl)]
            k_each = max(2, (max(3, args.steps) + n_fl - 1) // n_fl)     # at least `steps` frames in all: the timed region includes the
                                                                          # pipeline's fill (first H2D) and drain (last D2H), amortised over them

            def run_frames(i, k):
                torch.cuda.set_device(local_rank)
                for _ in range(k):
                    trks[i].tpc_track_timeframe_host(*host, n=n, outputs=houts[i], stream=streams[i])

            def run_all(k):
                th = [threading.Thread(target=run_frames, args=(i, k)) for i in range(n_fl)]
                for t_ in th:
                    t_.start()
                for t_ in th:
                    t_.join()

            run_all(1)                                   # warm-up
            barrier()
            e0.record(streams[0])
            run_all(k_each)
            for s_ in streams[1:]:
                streams[0].wait_stream(s_)
            e1.record(streams[0])
            barrier()
            k_e2e = k_each * n_fl
            ms = replicas.max_over_ranks(e0.elapsed_time(e1) / k_e2e, world, device=dev)
            k = int(houts[0][0].n_tracks[0]); h = int(houts[0][0].n_track_hits[0])
            d2h = 16 + k * (8 + 5 * 4 + 7 * 4 + 36) + 4 * h
            for t_ in trks:
                t_.close()
            return {"value": n_all / (float(ms) * 1e-3), "unit": "clusters/s", "ms_per_step": float(ms),
                    "h2d_bytes_per_step": 12 * n, "d2h_bytes_per_step": d2h, "steps": k_e2e, "frames_in_flight": n_fl}

        n_fl = max(1, args.e2e_inflight)
        e2e = measure_e2e(n_fl)                          # the headline: frames buffered the way a processing node runs (copies of one frame under the kernels of another)
        if n_fl != 1:                                    # ... and the latency-bound figure beside it: one frame at a time
            one = measure_e2e(1)
            e2e["one_frame_in_flight"] = {k: one[k] for k in ("value", "ms_per_step", "steps")}

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return 0

    # ---- per-kernel rooflines; `roofline` = the dominant kernel's ----
    peak, peak_src = _peaks()
    if cluster_finder:
        cluster_finder.update({"peak": peak, "frac": round(cluster_finder["achieved"] / peak, 4)})
    clk = clocks.summary()
    mhz = clk["sm_mhz"] or clk["sm_max_mhz"] or 1965.0
    alu_derived = SM_COUNT * SMSP_PER_SM * LANES * mhz * 1e6 / 1e12          # T lane-instructions / s at the clock under load
    alu_peak = alu_measured[0] / 1e12                                        # measured on this GPU in this run
    alu_src = (f"measured: tpc_selftest_alu_peak, dependency-free scalar FMUL/FADD streams on all SMs, no FMA contraction "
               f"({alu_peak:.2f} T lane-inst/s = {alu_peak / alu_derived:.3f} of 148 SMs x 4 schedulers x 32 lanes x {mhz:.0f} MHz); "
               f"the same arithmetic issued as packed f32x2 FFMA2 runs at {alu_measured[1] / 1e12:.2f} T fp32 op/s")
    total_step_ms = sum(step_acc.values())
    traffic = _ncu_traffic() if (cid == 3 and args.seed == 1 and not args.frame_us and args.follower == 0) else {}
    kernels = {}
    for k, ms in step_acc.items():
        row = {"ms": round(ms, 4), "share_of_step": round(ms / total_step_ms, 4)}
        if k in ALGO_BYTES_PER_CLUSTER and ms > 0:
            a = ALGO_BYTES_PER_CLUSTER[k] * n / (ms * 1e-3) / 1e9
            row.update({"bound": "hbm", "achieved": round(a, 1), "peak": peak, "unit": "GB/s", "frac": round(a / peak, 4),
                        "algo_bytes_per_cluster": ALGO_BYTES_PER_CLUSTER[k]})
        elif k in TRACKLET_PHASES and ms > 0:
            w = work[TRACKLET_PHASES[k]]
            inst = (ALGO_LANE_INST_TRANSPORT * w["row_steps"] + ALGO_LANE_INST_UPDATE * w["updates"] +
                    (ALGO_LANE_INST_PER_CANDIDATE * w["candidates"] if "follow" in k else 0))
            a = inst / (ms * 1e-3) / 1e12
            row.update({"bound": "alu", "achieved": round(a, 3), "peak": round(alu_peak, 3), "unit": "T lane-inst/s",
                        "frac": round(a / alu_peak, 4), "units": w})
        t = _step_traffic(traffic, k)
        if t:
            row["traffic"] = t[0]
        kernels[k] = row
    dom = max(step_acc, key=step_acc.get)
    t = _step_traffic(traffic, dom)
    roof = {"kernel": dom, "ms": step_acc[dom], "share_of_step": step_acc[dom] / total_step_ms,
            "traffic": t[0] if t else None,
            "traffic_source": (f"profiles/{NCU_TRAFFIC_CSV} (dram read + write bytes per launch, ncu --set full at commit {t[1]})" if t else None)}
    roof.update({k: v for k, v in kernels[dom].items() if k not in ("ms", "share_of_step", "traffic")})
    roof["peak_source"] = alu_src if roof.get("bound") == "alu" else peak_src
    if "bound" not in roof:
        roof.update({"bound": "hbm", "achieved": None, "peak": peak, "unit": "GB/s", "frac": None})
    # the whole constructor (seed + four phase kernels) against the same ALU peak
    c_ms = sum(step_acc.get(k, 0.0) for k in ("tracklet_init", *TRACKLET_PHASES))
    c_inst = (ALGO_LANE_INST_TRANSPORT * work["row_steps"] + ALGO_LANE_INST_UPDATE * work["updates"] +
              ALGO_LANE_INST_PER_CANDIDATE * (work["follow_up"]["candidates"] + work["follow_down"]["candidates"]))
    constructor = {"ms": round(c_ms, 4), "share_of_step": round(c_ms / total_step_ms, 4), "bound": "alu",
                   "achieved": round(c_inst / (c_ms * 1e-3) / 1e12, 3) if c_ms > 0 else None, "peak": round(alu_peak, 3),
                   "unit": "T lane-inst/s", "frac": round(c_inst / (c_ms * 1e-3) / 1e12 / alu_peak, 4) if c_ms > 0 else None,
                   "units": {k: work[k] for k in ("tracklets", "row_steps", "updates", "candidates")}}
    # the frame against the sum of its floors (HBM-bound steps at the measured copy bandwidth + the constructor at the ALU peak)
    floor_ms = sum(ALGO_BYTES_PER_CLUSTER.get(k, 0) for k in step_acc) * n / (peak * 1e9) * 1e3 + c_inst / (alu_peak * 1e12) * 1e3
    frame = {"sum_of_floors_ms": round(floor_ms, 3), "frac": round(floor_ms / total_step_ms, 4),
             "algorithmic_bytes_per_cluster": sum(ALGO_BYTES_PER_CLUSTER.get(k, 0) for k in step_acc)}

    cpu = None
    if not args.no_cpu_baseline:
        # (1) one core, a bounded sample (the paper's "speed-up vs 1 CPU core" convention)
        cn, cdt, _ = _cpu_oracle_run(cid, args.seed, args.cpu_sample_us)
        sample = (f"{CONFIG_NAMES[cid]} generator, seed {args.seed}, frame cut to {args.cpu_sample_us:g} us ({cn} clusters)"
                  if cid >= 2 else f"{CONFIG_NAMES[cid]} ({cn} clusters)")
        one_core = {"value": cn / cdt, "unit": "clusters/s", "cores": 1, "kind": "oracle", "sample": sample, "seconds": cdt}
        cpu = dict(one_core)
        if cfg.n_sectors > 1:
            # (2) all host cores (the unchanged oracle, one call per sector from a thread pool), on the
            # WHOLE frame the GPU arm timed -- the same configuration, about 20 s for a 10 ms frame on 16 cores
            whole = bool(args.cpu_whole_frame) and not args.frame_us
            an, adt, athreads, atracks = _cpu_oracle_run_all_cores(cid, args.seed, args.cpu_sample_us, tf=tf if whole else None)
            cpu = {"value": an / adt, "unit": "clusters/s", "cores": athreads, "host_cpus": os.cpu_count(), "cpu_model": _cpu_model(),
                   "kind": "oracle", "how": "the unchanged oracle, one call per sector from a thread pool",
                   "sample": (f"the whole frame the GPU arm timed ({an} clusters, same configuration)" if whole else sample),
                   "same_config": whole, "seconds": adt, "n_tracks": atracks, "one_core": one_core}

    line = {"metric": "tpc_clusters_tracked_per_s", "value": value, "unit": "clusters/s", "n_gpus": world,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True,
            "scaling": "strong" if by_sector else "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": CONFIG_NAMES[cid] + (f" (frame cut to {args.frame_us:g} us)" if args.frame_us else ""),
                       "n_clusters_rank0": n, "n_clusters_all_ranks": int(n_all), "n_collisions": tf.n_collisions,
                       "n_tracks": n_tracks, "n_track_hits": n_track_hits, "status": status, "seed": args.seed,
                       "parallelism": (f"one time frame cut by sector across {args.shard_of or world} GPU(s) (sectors {sector_range[0]}..{sector_range[1] - 1} on rank 0), "
                                       "no collective inside the tracking" if by_sector else f"{world} independent time frame(s), one per GPU"), "arena_gb": round(arena_gb, 2),
                       "l2": "inputs and scratch are larger than L2 (no flush needed)" if n * 12 > 2.5e8 else
                             "working set may fit L2 (small config)", "gen_seconds": round(t_gen, 1)},
            "clocks": clocks.summary(), "e2e": e2e, "gpu_launches": launches,
            "step_ms": {k: round(v, 4) for k, v in step_acc.items()}, "kernels": kernels,
            "tracklet_constructor": constructor, "frame_vs_floors": frame, "rare_paths": work.get("rare_paths"), "merge": merge,
            "cluster_finder": cluster_finder, "graph_replay": graph_replay,
            "roofline": roof, "cpu_baseline": cpu}
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
