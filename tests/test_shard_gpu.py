"""Sector sharding on the CUDA path (paper_2102_08862_b200/shard.py): the tracks of the shards
of ONE frame, each tracked by its own `tpc_track_timeframe` call as a rank of `bench.py --shard sectors` would, put
together are the whole frame's tracks -- same seeds, hit lists, parameters and covariances, bit for bit.  One GPU: the
shards run one after the other (they are independent; nothing waits on anything).
"""
from __future__ import annotations

import numpy as np
import pytest

from paper_2102_08862_b200 import gen, shard

pytestmark = pytest.mark.gpu
N_ROWS = 152
FIELDS = ("x", "y", "z_rel", "time_ref", "sin_phi", "dzds", "q_pt")


def _track(T, torch, tf, cfg, sel=None):
    row, pad, time = (tf.row, tf.pad, tf.time) if sel is None else (tf.row[sel], tf.pad[sel], tf.time[sel])
    n = int(row.shape[0])
    trk = T.Tracker(T.default_geometry(36, tf.max_time_bin), T.default_params(cfg.sigma_y_cm, cfg.sigma_z_cm, max_clusters=max(n, 1)))
    d = [torch.from_numpy(np.ascontiguousarray(a, np.float32)).to(trk.device) for a in (row, pad, time)]
    out = trk.tpc_track_timeframe(*d, n=n)
    torch.cuda.synchronize()
    k, nh = int(out.n_tracks[0]), int(out.n_track_hits[0])
    assert int(out.status[0]) == 0
    res = dict(seed=out.seed_hit[:k].cpu().numpy(), n_hits=out.n_hits[:k].cpu().numpy(), off=out.hit_offset[:k].cpu().numpy(),
               hits=out.hit_index[:nh].cpu().numpy(), sector=out.sector[:k].cpu().numpy(), cov=out.cov9[:k].cpu().numpy(),
               par=np.stack([getattr(out, f)[:k].cpu().numpy() for f in FIELDS], axis=1))
    trk.close()
    if sel is not None:
        res["seed"] = shard.global_index(sel, res["seed"]); res["hits"] = shard.global_index(sel, res["hits"])
    return res


@pytest.mark.parametrize("cid,seed,us,world", [(1, 4, None, 4), (3, 5, 120.0, 3), (4, 2, 100.0, 8)])
def test_the_shards_tracks_put_together_are_the_whole_frames_tracks(cid, seed, us, world):
    import torch
    from paper_2102_08862_b200 import tracker as T
    cfg = gen.preset(cid, seed) if us is None else gen.preset(cid, seed, us)
    tf = gen.generate(cfg, want_truth=False)
    whole = _track(T, torch, tf, cfg)
    ranges = shard.sector_ranges(36, world, shard.sector_histogram(tf.row, 36, N_ROWS))
    parts = []
    for lo, hi in ranges:
        sel = shard.shard_indices(tf.row, N_ROWS, lo, hi)
        p = _track(T, torch, tf, cfg, sel)
        assert np.all((p["sector"] >= lo) & (p["sector"] < hi))
        parts.append(p)
    assert len(whole["seed"]) > 500 and sum(len(p["seed"]) for p in parts) == len(whole["seed"])
    seed_s = np.concatenate([p["seed"] for p in parts]); nh_s = np.concatenate([p["n_hits"] for p in parts])
    par_s = np.concatenate([p["par"] for p in parts]); cov_s = np.concatenate([p["cov"] for p in parts])
    hits_s = np.concatenate([p["hits"] for p in parts])
    off_s = np.concatenate([[0], np.cumsum(nh_s)[:-1]])
    ow, os_ = np.argsort(whole["seed"], kind="stable"), np.argsort(seed_s, kind="stable")
    np.testing.assert_array_equal(whole["seed"][ow], seed_s[os_])
    np.testing.assert_array_equal(whole["n_hits"][ow], nh_s[os_])
    assert np.array_equal(whole["par"][ow].view(np.uint32), par_s[os_].view(np.uint32))
    assert np.array_equal(whole["cov"][ow].view(np.uint32), cov_s[os_].view(np.uint32))
    for a, b in zip(ow, os_):
        n = whole["n_hits"][a]
        assert np.array_equal(whole["hits"][whole["off"][a]:whole["off"][a] + n], hits_s[off_s[b]:off_s[b] + n])
