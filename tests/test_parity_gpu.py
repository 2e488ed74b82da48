"""Parity of the CUDA path (through the C-ABI) with the oracle, element by element on the same seeded inputs.

Bit-exact: cleaned neighbour links, start hits, tracklet row->hit tables, track hit lists.  Fits: y, z within
1e-3 cm, q/pT within 1e-4 relative (BASELINE.json L5).  Run on the B200 box: ``pytest -m gpu``.
"""
import numpy as np
import pytest

from helpers import N_ROWS, clusters_from_xyz, concat, row_x
from paper_2102_08862_b200 import gen
import parity_util as PU

pytestmark = pytest.mark.gpu


def _frame(cid, seed, frame_us=None, **kw):
    c = gen.preset(cid, seed, frame_us)
    for k, v in kw.items():
        setattr(c, k, v)
    return c, gen.generate(c)


def _both(tf, cfg, time=None, tmax=None, **overrides):
    time = tf.time if time is None else time
    tmax = tf.max_time_bin if tmax is None else tmax
    g = PU.run_gpu(tf.row, tf.pad, time, cfg.n_sectors, tmax, cfg.sigma_y_cm, cfg.sigma_z_cm, **overrides)
    o = PU.run_oracle(tf.row, tf.pad, time, cfg.n_sectors, tmax, cfg.sigma_y_cm, cfg.sigma_z_cm, **overrides)
    return g, o


@pytest.mark.parametrize("seed", [1, 2, 3])
def test_config0_single_sector(seed):
    cfg, tf = _frame(0, seed)
    g, o = _both(tf, cfg)
    rep = PU.compare(g, o)
    assert rep["n_tracks"] > 50 and rep["n_links"] > 1000
    assert rep["track_par_bit_identical"] and rep["tracklet_par_bit_identical"]


@pytest.mark.parametrize("seed", [1, 2, 3])
def test_config1_full_tpc(seed):
    cfg, tf = _frame(1, seed)
    g, o = _both(tf, cfg)
    rep = PU.compare(g, o)
    assert rep["n_tracks"] > 5000
    assert rep["track_par_bit_identical"] and rep["tracklet_par_bit_identical"] and rep["track_cov_bit_identical"]


@pytest.mark.parametrize("cid,seed", [(2, 1), (3, 2), (4, 1), (4, 3)])
def test_continuous_readout_short_frames(cid, seed):
    """configs[2..4] with the frame cut to 150 us (7-8 overlapping collisions): same generator, oracle-sized."""
    cfg, tf = _frame(cid, seed, frame_us=150.0)
    g, o = _both(tf, cfg)
    rep = PU.compare(g, o)
    assert rep["n_tracks"] > 1000


@pytest.mark.parametrize("cid,seed,frame_us", [(0, 1, None), (1, 2, None), (2, 1, 150.0), (4, 3, 150.0)])
def test_row_synchronous_follower_matches_the_oracle(cid, seed, frame_us):
    """params.follower = 1: the lock-step follower with bulk-copy-staged rows (csrc/follow_rows.cuh) -- not the default, kept
    for A/B -- gives the same links, tracklets, tracks and fits, bit for bit; nearly every search runs on the staged rows."""
    cfg, tf = _frame(cid, seed, frame_us)
    g, o = _both(tf, cfg, follower=1)
    rep = PU.compare(g, o)
    assert rep["track_par_bit_identical"] and rep["tracklet_par_bit_identical"] and rep["track_cov_bit_identical"]
    w = g["work"]
    searches = w["follow_up"]["row_steps"] + w["follow_down"]["row_steps"]
    assert searches > 1000 and w["rare_paths"]["searches_in_global_memory"] < 0.05 * searches


def test_row_synchronous_follower_other_cuts_and_grids():
    cfg, tf = _frame(0, 6)
    for kw in (dict(seed_min_hits=5, miss_limit=4, min_hits=20, chi2_cut=4.0), dict(grid_time_bins=2, grid_pad_bins=3),
               dict(grid_time_bins=16, grid_pad_bins=64), dict(miss_limit=30, win_slope=0.2)):
        g = PU.run_gpu(tf.row, tf.pad, tf.time, 1, tf.max_time_bin, follower=1, **kw)
        okw = {k: v for k, v in kw.items() if not k.startswith("grid_")}
        o = PU.run_oracle(tf.row, tf.pad, tf.time, 1, tf.max_time_bin, **okw)
        PU.compare(g, o)


def test_rare_paths_of_the_constructor_are_taken_and_agree():
    """The refit's replay (a failed transport after a hole) and the refit that fails before its first update (the up
    pass's state is the result) are rare; this input takes both (device counters), and parity holds on it."""
    cfg, tf = _frame(1, 2, pt_min=0.05)
    g, o = _both(tf, cfg)
    rep = PU.compare(g, o)
    assert rep["track_par_bit_identical"] and rep["tracklet_par_bit_identical"] and rep["track_cov_bit_identical"]
    rare = g["work"]["rare_paths"]
    assert rare["refit_replays"] >= 1 and rare["refits_without_update"] >= 20, rare


def test_time_coordinate_at_the_end_of_a_10ms_frame():
    """fp32 time values near 5e4 bins (ulp 2^-8 bin): all z arithmetic is on differences of raw time values."""
    cfg, tf = _frame(3, 5, frame_us=100.0)
    time = (tf.time.astype(np.float64) + 49000.0).astype(np.float32)
    g, o = _both(tf, cfg, time=time, tmax=tf.max_time_bin + 49000.0)
    rep = PU.compare(g, o)
    assert rep["n_tracks"] > 500


@pytest.mark.parametrize("grid_time_bins,grid_pad_bins", [(1, 1), (3, 2), (16, 8), (2, 5), (4, 64)])
def test_grid_bin_width_does_not_change_results(grid_time_bins, grid_pad_bins):
    """The grid only accelerates (BASELINE.json L5 (b)): any bin shape gives the oracle's links and tracks."""
    cfg, tf = _frame(0, 4)
    g = PU.run_gpu(tf.row, tf.pad, tf.time, 1, tf.max_time_bin, grid_time_bins=grid_time_bins, grid_pad_bins=grid_pad_bins)
    o = PU.run_oracle(tf.row, tf.pad, tf.time, 1, tf.max_time_bin)
    PU.compare(g, o)


def test_other_cuts():
    cfg, tf = _frame(0, 6)
    g, o = _both(tf, cfg, seed_min_hits=5, miss_limit=4, min_hits=20, chi2_cut=4.0)
    PU.compare(g, o)


def test_empty_and_tiny_inputs():
    e = np.zeros(0, np.float32)
    g = PU.run_gpu(e, e, e, 36, 487.0)
    assert int(g["n_tracks"][0]) == 0 and int(g["n_track_hits"][0]) == 0 and int(g["status"][0]) == 0
    assert int(g["n_tracklets"][0]) == 0
    one = clusters_from_xyz([5], [0.3], [100.0])
    g = PU.run_gpu(*one, 1, 487.0)
    o = PU.run_oracle(*one, 1, 487.0)
    PU.compare(g, o)
    assert int(g["n_tracks"][0]) == 0


def test_invalid_clusters_are_ignored_and_flagged():
    cfg, tf = _frame(0, 2)
    row, pad, time = tf.row.copy(), tf.pad.copy(), tf.time.copy()
    row[::97] = 152.0            # beyond the single sector
    row[5::101] += 0.5           # not an integer
    pad[3::89] = 400.0
    pad[7::83] = -0.75
    time[11::79] = -1.0
    time[13::73] = tf.max_time_bin + 10.0
    g = PU.run_gpu(row, pad, time, 1, tf.max_time_bin)
    o = PU.run_oracle(row, pad, time, 1, tf.max_time_bin)
    PU.compare(g, o)
    assert int(g["status"][0]) & 8
    assert o.stats["invalid_clusters"] > 500


@pytest.mark.parametrize("copies", [2, 6, 9])
def test_duplicate_hits_tie_break_on_original_index(copies):
    """Exact duplicates of whole tracks: every chi2 / distance tie must go to the lowest original index
    (6 copies fill the finder's 6 candidate slots per row exactly, 9 overflow them -> generic path)."""
    rows = np.arange(N_ROWS)
    x = row_x(rows)
    parts = []
    for i in range(4):
        y = (-0.1 + 0.06 * i) * x
        z = 100.0 + 0.3 * i * (x - 85.0)
        p = clusters_from_xyz(rows, y, z)
        parts += [p] * copies                             # each track several times
    row, pad, time = concat(parts)
    rng = np.random.default_rng(3)
    perm = rng.permutation(row.size)
    row, pad, time = row[perm], pad[perm], time[perm]
    g = PU.run_gpu(row, pad, time, 1, 487.0)
    o = PU.run_oracle(row, pad, time, 1, 487.0)
    rep = PU.compare(g, o)
    assert rep["n_tracks"] >= 4
    assert g["work"]["rare_paths"]["search_ties"] > 0          # the follower's exact-tie path ran


def test_runs_are_deterministic_including_output_order():
    cfg, tf = _frame(1, 7)
    a = PU.run_gpu(tf.row, tf.pad, tf.time, 36, tf.max_time_bin)
    b = PU.run_gpu(tf.row, tf.pad, tf.time, 36, tf.max_time_bin)
    k, h = int(a["n_tracks"][0]), int(a["n_track_hits"][0])
    assert k == int(b["n_tracks"][0])
    for name in ("seed_hit", "n_hits", "hit_offset", "q_pt", "y"):
        np.testing.assert_array_equal(a[name][:k], b[name][:k])
    np.testing.assert_array_equal(a["hit_index"][:h], b["hit_index"][:h])
    nt = int(a["n_tracklets"][0])
    np.testing.assert_array_equal(a["tracklet_seed"][:nt], b["tracklet_seed"][:nt])


def test_capacity_overflow_sets_status_and_keeps_a_valid_prefix():
    import torch
    from paper_2102_08862_b200 import tracker as T
    cfg, tf = _frame(0, 1)
    full = PU.run_gpu(tf.row, tf.pad, tf.time, 1, tf.max_time_bin)
    k = int(full["n_tracks"][0])
    g = T.default_geometry(1, tf.max_time_bin)
    p = T.default_params(max_clusters=tf.n)
    trk = T.Tracker(g, p)
    d = [torch.from_numpy(a).cuda() for a in (tf.row, tf.pad, tf.time)]
    outs = trk.alloc_outputs(tf.n, max_tracks=10, max_track_hits=500)
    out = trk.tpc_track_timeframe(*d, outputs=outs)
    torch.cuda.synchronize()
    assert int(out.status[0]) & 2 and int(out.status[0]) & 4
    assert int(out.n_tracks[0]) == k
    np.testing.assert_array_equal(out.seed_hit.cpu().numpy(), full["seed_hit"][:10])
    trk.close()
    p = T.default_params(max_clusters=tf.n)
    p.max_tracklets = 100
    trk = T.Tracker(g, p)
    out = trk.tpc_track_timeframe(*d)
    torch.cuda.synchronize()
    assert int(out.status[0]) & 1
    trk.close()


def test_host_entry_point_matches_device_entry_point():
    import torch
    from paper_2102_08862_b200 import tracker as T
    cfg, tf = _frame(1, 2)
    ref = PU.run_gpu(tf.row, tf.pad, tf.time, 36, tf.max_time_bin, taps=False)
    g = T.default_geometry(36, tf.max_time_bin)
    p = T.default_params(max_clusters=tf.n)
    p.host_staging = 1
    trk = T.Tracker(g, p)
    h = [torch.from_numpy(a).pin_memory() for a in (tf.row, tf.pad, tf.time)]
    out = trk.tpc_track_timeframe_host(*h)
    k, nh = int(out.n_tracks[0]), int(out.n_track_hits[0])
    assert k == int(ref["n_tracks"][0]) and nh == int(ref["n_track_hits"][0])
    for name in ("seed_hit", "sector", "first_row", "last_row", "n_hits", "hit_offset", "x", "y", "z_rel", "time_ref",
                 "sin_phi", "dzds", "q_pt", "cov9"):
        np.testing.assert_array_equal(getattr(out, name).numpy()[:k], ref[name][:k], err_msg=name)
    np.testing.assert_array_equal(out.hit_index.numpy()[:nh], ref["hit_index"][:nh])
    trk.close()


def test_arena_plan_reuses_memory_across_steps():
    from paper_2102_08862_b200 import tracker as T
    g = T.default_geometry(36, 2000.0)
    trk = T.Tracker(g, T.default_params(max_clusters=1_000_000))
    plan = trk.arena_plan()
    by = {a["name"]: a for a in plan}
    total = sum(a["bytes"] for a in plan)
    assert trk.arena_bytes < total
    # no two arrays alive in the same step overlap in memory
    for i, a in enumerate(plan):
        for b in plan[i + 1:]:
            if a["first_step"] <= b["last_step"] and b["first_step"] <= a["last_step"]:
                assert a["offset"] + a["bytes"] <= b["offset"] or b["offset"] + b["bytes"] <= a["offset"], (a, b)
    # the selector's claim array lives in memory that earlier steps used
    c = by["selector_claim(u64)"]
    assert any(a["last_step"] < c["first_step"] and a["offset"] < c["offset"] + c["bytes"] and c["offset"] < a["offset"] + a["bytes"]
               for a in plan)
    trk.close()


def test_fast_sqrt_rcp_are_ieee_exact_exhaustively():
    """The constructor replaces sqrtf() and 1.0f / x by range-restricted refinement sequences (csrc/tracklet.cuh); they
    must be bit-identical to the IEEE results the oracle computes, for EVERY fp32 operand of their ranges."""
    from paper_2102_08862_b200 import tracker as T
    bad_sqrt, bad_rcp = T.tpc_selftest_fast_math()
    assert (bad_sqrt, bad_rcp) == (0, 0)


_FULL = {}


def _full_frame(cid):
    """The full frame of configs[cid], seed 1 (the one bench.py times); one multi-GB frame in host memory at a time."""
    if cid not in _FULL:
        _FULL.clear()
        c = gen.preset(cid, 1)
        _FULL[cid] = (c, gen.generate(c, want_truth=False))
    return _FULL[cid]


@pytest.mark.parametrize("cid", [2, 3, 4])
def test_whole_frame_oracle_parity_at_full_size(cid):
    """BASELINE.json L5 "GPU tracks identical to the oracle ... on all five configs": configs[2] (2 ms, 4e7 clusters),
    configs[3] and configs[4] (10 ms, 1.6e8 clusters) at FULL size, in the launch configuration bench.py times (default
    parameters; the link / start-hit / tracklet-summary taps add three small kernels' worth of writes).  The oracle runs
    unchanged, once per sector from a thread pool (sectors are independent -- reading A16 -- and a per-sector sub-frame
    keeps the cluster order, so original-index tie-breaks and tracklet ids map through the selection).  Compared bit
    for bit, over the WHOLE frame: every cleaned link and start hit, every tracklet's (seed, n_hits, 7 parameters),
    every track's hit list, rows, parameters and covariance.  (The tracklets' row->hit tables are 10 GB at this size;
    they are compared in full on configs[0], [1] and the short frames -- here the tracklet parameters, which depend on
    every attached hit in order, stand in for them.)"""
    import torch
    from paper_2102_08862_b200 import tracker as T
    cfg, tf = _full_frame(cid)
    n = tf.n
    assert n > (3e7 if cid == 2 else 1.2e8)
    g = T.default_geometry(cfg.n_sectors, tf.max_time_bin)
    trk = T.Tracker(g, T.default_params(cfg.sigma_y_cm, cfg.sigma_z_cm, max_clusters=n))
    d = [torch.from_numpy(a).to(trk.device) for a in (tf.row, tf.pad, tf.time)]
    outs = trk.alloc_outputs(n, taps=True, tap_row_hit=False)
    out = trk.tpc_track_timeframe(*d, n=n, outputs=outs)
    torch.cuda.synchronize()
    gpu = {k: (v.cpu().numpy() if v is not None else None) for k, v in out.__dict__.items()}
    trk.close()
    del d, out, outs
    torch.cuda.empty_cache()
    k, nh, status = int(gpu["n_tracks"][0]), int(gpu["n_track_hits"][0]), int(gpu["status"][0])
    assert status == 0 and k > (2e5 if cid == 2 else 1e6)
    orc = PU.run_oracle_per_sector(tf.row, tf.pad, tf.time, cfg.n_sectors, tf.max_time_bin, cfg.sigma_y_cm, cfg.sigma_z_cm)
    rep = PU.compare_whole_frame(gpu, orc)
    assert rep["n_tracks_compared"] == k == rep["n_tracks_oracle"]
    assert rep["n_track_hits_compared"] == nh
    assert rep["n_tracklets_compared"] == int(gpu["n_tracklets"][0])
    assert rep["n_links_compared"] == n
    # properties that hold at any size (hit rows ascend inside a track, a hit in at most one track, offsets are the scan)
    n_hits, off, hit_index = gpu["n_hits"][:k], gpu["hit_offset"][:k], gpu["hit_index"][:nh]
    assert n_hits.min() >= 30 and n_hits.max() <= N_ROWS
    np.testing.assert_array_equal(off, np.concatenate([[0], np.cumsum(n_hits[:-1], dtype=np.int64)]))
    assert np.bincount(hit_index, minlength=n).max() == 1, "a hit belongs to more than one track"
    hrow = tf.row[hit_index].astype(np.int64)
    assert np.array_equal(hrow // N_ROWS, np.repeat(gpu["sector"][:k], n_hits)), "a track holds hits of another sector"
    r_in = hrow % N_ROWS
    inner = np.ones(nh, bool); inner[off] = False
    assert np.all(r_in[inner] > r_in[np.nonzero(inner)[0] - 1]), "hit rows must ascend inside a track"
    assert np.array_equal(r_in[off], gpu["first_row"][:k]) and np.array_equal(r_in[off + n_hits - 1], gpu["last_row"][:k])


def test_empty_and_sparse_frames_on_the_10ms_grid_are_cheap():
    """2.8e8 grid bins and (almost) nothing in them: the runs of empty bins are filled by whole CTAs, not by one thread
    (a single thread writing every bin took seconds); results still equal the oracle's."""
    import time as _time
    import torch
    from paper_2102_08862_b200 import tracker as T
    cfg, tf = _frame(0, 3)                                     # 1.3e4 clusters of one sector ...
    row = tf.row + np.float32(17 * N_ROWS)                      # ... moved to sector 17 of the 36-sector, 10 ms geometry
    time = (tf.time.astype(np.float64) + 30000.0).astype(np.float32)
    tmax = 50485.0
    g = T.default_geometry(36, tmax)
    trk = T.Tracker(g, T.default_params(max_clusters=tf.n))
    d = [torch.from_numpy(np.ascontiguousarray(a, np.float32)).to(trk.device) for a in (row, tf.pad, time)]
    e = torch.zeros(0, dtype=torch.float32, device=trk.device)
    for clusters, n in ((d, tf.n), ([e, e, e], 0)):
        outs = trk.alloc_outputs(max(n, 1))
        trk.tpc_track_timeframe(*clusters, n=n, outputs=outs)   # warm-up
        torch.cuda.synchronize()
        t0 = _time.perf_counter()
        out = trk.tpc_track_timeframe(*clusters, n=n, outputs=outs)
        torch.cuda.synchronize()
        assert _time.perf_counter() - t0 < 0.05, "a sparse frame on the long-frame grid must not take longer than a full one"
        assert int(out.status[0]) == 0
    trk.close()
    gres = PU.run_gpu(row, tf.pad, time, 36, tmax)
    ores = PU.run_oracle(row, tf.pad, time, 36, tmax)
    assert PU.compare(gres, ores)["n_tracks"] > 50
