"""Sector sharding of ONE frame across ranks (paper_2102_08862_b200/shard.py), on CPU:
the index arithmetic, and two `gloo` ranks that each track their sectors (with the oracle standing in for the GPU path: this
is a test) and gather the tracks -- the concatenation must be the whole frame's result, index for index and bit for bit.
"""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2102_08862_b200 import gen, shard

N_ROWS = 152


def test_sector_ranges_cover_are_contiguous_and_balanced():
    for n_sec, world in ((36, 1), (36, 2), (36, 4), (36, 8), (36, 5), (36, 36), (18, 4), (1, 1)):
        r = shard.sector_ranges(n_sec, world)
        assert len(r) == world and r[0][0] == 0 and r[-1][1] == n_sec
        assert all(a[1] == b[0] for a, b in zip(r, r[1:]))
        sizes = [hi - lo for lo, hi in r]
        assert min(sizes) >= 1 and max(sizes) - min(sizes) <= 1, (n_sec, world, sizes)
    r = shard.sector_ranges(4, 6)                                      # more ranks than sectors: the surplus ranks get nothing
    assert r == [(0, 1), (1, 2), (2, 3), (3, 4), (4, 4), (4, 4)]
    w = np.ones(36); w[:9] = 7.0                                       # a hot quarter of the TPC: cuts follow the cluster counts
    r = shard.sector_ranges(36, 4, w)
    loads = [w[lo:hi].sum() for lo, hi in r]
    assert r[0][1] < 9 and max(loads) <= 1.3 * w.sum() / 4 and r[-1][1] == 36
    with pytest.raises(ValueError):
        shard.sector_ranges(0, 2)
    with pytest.raises(ValueError):
        shard.sector_ranges(36, 2, np.ones(35))


def test_shard_indices_partition_the_valid_clusters_in_order():
    tf = gen.generate(gen.preset(1, 3), want_truth=False)
    row = tf.row.copy()
    row[[5, 77]] = [-1.0, 36 * N_ROWS]                                 # two clusters outside the geometry
    row[100] = 40.5
    hist = shard.sector_histogram(row, 36, N_ROWS)
    assert hist.sum() == tf.n - 3 and hist.shape == (36,)
    parts = [shard.shard_indices(row, N_ROWS, lo, hi) for lo, hi in shard.sector_ranges(36, 4, hist)]
    allv = np.concatenate(parts)
    assert allv.size == tf.n - 3 and np.unique(allv).size == allv.size and not np.isin([5, 77, 100], allv).any()
    for (lo, hi), p in zip(shard.sector_ranges(36, 4, hist), parts):
        assert np.all(np.diff(p) > 0) and p.size == hist[lo:hi].sum()
        assert np.all((row[p] // N_ROWS >= lo) & (row[p] // N_ROWS < hi))
    sel = parts[1]
    np.testing.assert_array_equal(shard.global_index(sel, np.array([0, -1, 2, sel.size - 1])), [sel[0], -1, sel[2], sel[-1]])


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out_dir):
    import oracle
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world), LOCAL_RANK=str(rank))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        cfg = gen.preset(1, 2)
        cfg.fixed_tracks = 1500
        tf = gen.generate(cfg)                                         # every rank holds the same frame (same seed)
        g, p = oracle.default_geometry(36, tf.max_time_bin), oracle.default_params(cfg.sigma_y_cm, cfg.sigma_z_cm)
        lo, hi = shard.sector_ranges(36, world, shard.sector_histogram(tf.row, 36, N_ROWS))[rank]
        sel = shard.shard_indices(tf.row, N_ROWS, lo, hi)
        r = oracle.track(g, p, tf.row[sel], tf.pad[sel], tf.time[sel])
        seed = torch.from_numpy(shard.global_index(sel, r.tr_seed))
        hits = torch.from_numpy(shard.global_index(sel, r.tr_hit_index))
        par = torch.from_numpy(np.ascontiguousarray(r.tr_par))
        nh = torch.from_numpy(np.ascontiguousarray(r.tr_n_hits))
        g_seed, lens = shard.all_gather_ragged(seed, world)
        g_hits, hit_lens = shard.all_gather_ragged(hits, world)
        g_par, _ = shard.all_gather_ragged(par, world)
        g_nh, _ = shard.all_gather_ragged(nh, world)
        assert lens[rank] == len(r.tr_seed) and hit_lens[rank] == len(r.tr_hit_index)
        torch.save({"seed": g_seed, "hits": g_hits, "par": g_par, "nh": g_nh, "lens": lens, "range": (lo, hi), "n_sel": int(sel.size)},
                   os.path.join(out_dir, f"s{rank}.pt"))
    finally:
        dist.destroy_process_group()


@pytest.mark.timeout(600)
def test_two_gloo_ranks_track_their_sectors_and_the_gathered_tracks_are_the_whole_frames(tmp_path):
    import oracle
    world = 2
    mp.spawn(_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    r = [torch.load(os.path.join(str(tmp_path), f"s{k}.pt")) for k in range(world)]
    for key in ("seed", "hits", "par", "nh"):
        assert torch.equal(r[0][key], r[1][key]), key                  # every rank holds the same gathered result
    assert r[0]["range"][1] == r[1]["range"][0] and r[0]["range"][0] == 0 and r[1]["range"][1] == 36
    cfg = gen.preset(1, 2)
    cfg.fixed_tracks = 1500
    tf = gen.generate(cfg)
    assert r[0]["n_sel"] + r[1]["n_sel"] == tf.n and min(r[0]["n_sel"], r[1]["n_sel"]) > 0.4 * tf.n
    whole = oracle.track(oracle.default_geometry(36, tf.max_time_bin), oracle.default_params(cfg.sigma_y_cm, cfg.sigma_z_cm),
                         tf.row, tf.pad, tf.time)
    assert len(whole.tr_seed) > 1000 and sum(r[0]["lens"]) == len(whole.tr_seed)
    order_w, order_s = np.argsort(whole.tr_seed, kind="stable"), np.argsort(r[0]["seed"].numpy(), kind="stable")
    np.testing.assert_array_equal(whole.tr_seed[order_w], r[0]["seed"].numpy()[order_s])
    np.testing.assert_array_equal(whole.tr_n_hits[order_w], r[0]["nh"].numpy()[order_s])
    assert np.array_equal(whole.tr_par[order_w], r[0]["par"].numpy()[order_s])               # bit for bit
    off_s = np.concatenate([[0], np.cumsum(r[0]["nh"].numpy())[:-1]])
    hs = r[0]["hits"].numpy()
    for a, b in zip(order_w, order_s):
        n = whole.tr_n_hits[a]
        assert np.array_equal(whole.tr_hit_index[whole.tr_hit_offset[a]:whole.tr_hit_offset[a] + n], hs[off_s[b]:off_s[b] + n])
