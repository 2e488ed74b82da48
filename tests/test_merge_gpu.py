"""GPU parity of C7 (tpc_merge_tracks) against oracle/tpc_merge_oracle.cpp: the links are integer work -> bit-exact.

Both sides get THEIR OWN tracks (CUDA tracker -> CUDA merger, oracle tracker -> oracle merger); tracks are joined on
their seed id, links are compared as (seed of A -> seed of B).
"""
from __future__ import annotations

import ctypes as C

import numpy as np
import pytest

from paper_2102_08862_b200 import gen

pytestmark = pytest.mark.gpu


def _gpu_track_and_merge(tf, cfg, n_sectors=36, merge_params=None):
    import torch
    from paper_2102_08862_b200 import tracker as T
    n = tf.n
    trk = T.Tracker(T.default_geometry(n_sectors, tf.max_time_bin), T.default_params(cfg.sigma_y_cm, cfg.sigma_z_cm, max_clusters=max(n, 1)))
    d = [torch.from_numpy(np.ascontiguousarray(a, np.float32)).to(trk.device) for a in (tf.row, tf.pad, tf.time)]
    outs = trk.alloc_outputs(n)
    out = trk.tpc_track_timeframe(*d, n=n, outputs=outs)
    nxt, prv, root, n_links = trk.tpc_merge_tracks(outs, merge_params)
    torch.cuda.synchronize()
    k = int(out.n_tracks[0])
    res = dict(k=k, seed=out.seed_hit[:k].cpu().numpy(), next=nxt.cpu().numpy(), prev=prv.cpu().numpy(), root=root.cpu().numpy(),
               n_links=int(n_links[0]), launches=trk.last_merge_launches(), status=int(out.status[0]),
               sector=out.sector[:k].cpu().numpy(), first_row=out.first_row[:k].cpu().numpy(), last_row=out.last_row[:k].cpu().numpy())
    trk.close()
    return res


def _oracle_track_and_merge(tf, cfg, n_sectors=36, mp=None):
    import oracle
    from oracle import merge as M
    res = oracle.track(oracle.default_geometry(n_sectors, tf.max_time_bin), oracle.default_params(cfg.sigma_y_cm, cfg.sigma_z_cm),
                       tf.row, tf.pad, tf.time)
    mp = mp if mp is not None else M.default_merge_params(n_sectors)
    return res, M.merge(mp, res.tr_seed, res.tr_sector, res.tr_first_row, res.tr_last_row, res.tr_par)


def _as_seed_links(seed, idx):
    return np.where(idx >= 0, seed[np.maximum(idx, 0)], -1)


def _compare(g, res, mr):
    k = g["k"]
    assert g["status"] & 7 == 0
    assert k == len(res.tr_seed)
    go, oo = np.argsort(g["seed"], kind="stable"), np.argsort(res.tr_seed, kind="stable")
    np.testing.assert_array_equal(g["seed"][go], res.tr_seed[oo])
    for name, ref in (("next", mr.next), ("prev", mr.prev), ("root", mr.root)):
        np.testing.assert_array_equal(_as_seed_links(g["seed"], g[name][:k])[go], _as_seed_links(res.tr_seed, ref)[oo], err_msg=name)
    assert g["n_links"] == mr.n_links
    assert np.all(g["next"][k:] == -1) and np.all(g["prev"][k:] == -1) and np.all(g["root"][k:] == -1)
    assert g["launches"] >= 8


@pytest.mark.parametrize("seed", [1, 2, 3])
def test_merge_config1_full_tpc(seed):
    cfg = gen.preset(1, seed)
    tf = gen.generate(cfg)
    g = _gpu_track_and_merge(tf, cfg)
    res, mr = _oracle_track_and_merge(tf, cfg)
    _compare(g, res, mr)
    assert mr.n_links > 2000


@pytest.mark.parametrize("cid,seed,us", [(2, 1, 150.0), (4, 2, 100.0)])
def test_merge_continuous_readout_short_frames(cid, seed, us):
    """Several overlapping collisions: the time cells of the candidate index and the time_ref differences matter."""
    cfg = gen.preset(cid, seed, us)
    tf = gen.generate(cfg)
    g = _gpu_track_and_merge(tf, cfg)
    res, mr = _oracle_track_and_merge(tf, cfg)
    _compare(g, res, mr)
    assert mr.n_links > 500


def test_merge_other_cuts_and_row_window():
    from oracle import merge as M
    from paper_2102_08862_b200 import tracker as T
    cfg = gen.preset(1, 5)
    tf = gen.generate(cfg)
    g = _gpu_track_and_merge(tf, cfg, merge_params=T.MergeParams(0.7, 3.0, 0.02, 0.2, 4, 0))
    mp = M.default_merge_params(36)
    mp.cut_y_cm, mp.cut_z_cm, mp.cut_sin_phi, mp.cut_q_pt, mp.max_row_gap, mp.max_row_overlap = 0.7, 3.0, 0.02, 0.2, 4, 0
    res, mr = _oracle_track_and_merge(tf, cfg, mp=mp)
    _compare(g, res, mr)


def test_merge_single_sector_and_empty_frame():
    cfg = gen.preset(0, 1)
    tf = gen.generate(cfg)
    g = _gpu_track_and_merge(tf, cfg, n_sectors=1)
    assert g["k"] > 50 and g["n_links"] == 0 and np.all(g["next"] == -1)
    np.testing.assert_array_equal(g["root"][:g["k"]], np.arange(g["k"]))
    # empty frame through a 36-sector tracker
    import torch
    from paper_2102_08862_b200 import tracker as T
    trk = T.Tracker(T.default_geometry(36, 487.0), T.default_params(max_clusters=1))
    z = torch.zeros(0, dtype=torch.float32, device=trk.device)
    outs = trk.alloc_outputs(0)
    trk.tpc_track_timeframe(z, z, z, n=0, outputs=outs)
    nxt, prv, root, n_links = trk.tpc_merge_tracks(outs)
    torch.cuda.synchronize()
    assert int(n_links[0]) == 0 and bool((nxt == -1).all())
    trk.close()


def test_merge_rejects_bad_arguments():
    import torch
    from paper_2102_08862_b200 import tracker as T
    trk = T.Tracker(T.default_geometry(36, 487.0), T.default_params(max_clusters=1000))
    outs = trk.alloc_outputs(1000)
    z = torch.zeros(0, dtype=torch.float32, device=trk.device)
    trk.tpc_track_timeframe(z, z, z, n=0, outputs=outs)
    with pytest.raises(T.TpcError) as e:
        trk.tpc_merge_tracks(outs, T.MergeParams(0.0, 2.0, 0.05, 0.5, 12, 2))
    assert e.value.code == T.TPC_EINVAL
    assert trk.merge_scratch_bytes(outs[1].max_tracks) <= trk.arena_bytes
    # a track capacity whose scratch does not fit the arena is refused on the host
    big = T.Tracks.from_buffer_copy(outs[1])
    big.max_tracks = 2_000_000_000
    m = T.Merged(*(t.data_ptr() for t in (torch.empty(1, dtype=torch.int32, device=trk.device),) * 4))
    rc = trk.lib.tpc_merge_tracks(trk.handle, C.byref(T.default_merge_params()), C.byref(big), None, C.byref(m))
    assert rc == T.TPC_ENOMEM
    torch.cuda.synchronize()
    trk.close()
