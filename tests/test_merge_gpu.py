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
    outs = trk.alloc_outputs(n, hit_coords=True)
    out = trk.tpc_track_timeframe(*d, n=n, outputs=outs)
    nxt, prv, root, n_links = merged = trk.tpc_merge_tracks(outs, merge_params)
    launches_merge = trk.last_merge_launches()
    rf = trk.tpc_refit_chains(outs, merged)
    launches_refit = trk.last_merge_launches()
    vtx = trk.tpc_vertex_time(out.n_tracks, rf[3])
    torch.cuda.synchronize()
    k = int(out.n_tracks[0])
    nh = int(out.n_track_hits[0])
    hi = out.hit_index[:nh].cpu().numpy()
    hyt, hrow = out.hit_y_time[:nh].cpu().numpy(), out.hit_row[:nh].cpu().numpy()
    # the optional hit coordinates are those of hit_index: time verbatim, row, y = (pad - c_r) * pitch in fp32
    assert np.array_equal(hyt[:, 1], tf.time[hi]) and np.array_equal(hrow, (tf.row[hi].astype(np.int64) % 152).astype(np.uint8))
    npads = np.floor(2.0 * (85.0 + 1.07 * np.arange(152)) * np.tan(np.radians(10.0)) / 0.5)
    cr = (0.5 * (npads - 1)).astype(np.float32)
    assert np.array_equal(hyt[:, 0], (tf.pad[hi] - cr[hrow]) * np.float32(0.5))
    res = dict(k=k, vertex=tuple(t[:int(out.n_tracks[0])].cpu().numpy() for t in vtx), refit=tuple(t[:k].cpu().numpy() for t in rf), launches_refit=launches_refit, seed=out.seed_hit[:k].cpu().numpy(), next=nxt.cpu().numpy(), prev=prv.cpu().numpy(), root=root.cpu().numpy(),
               n_links=int(n_links[0]), launches=launches_merge, status=int(out.status[0]),
               sector=out.sector[:k].cpu().numpy(), first_row=out.first_row[:k].cpu().numpy(), last_row=out.last_row[:k].cpu().numpy())
    trk.close()
    return res


def _oracle_track_and_merge(tf, cfg, n_sectors=36, mp=None):
    import oracle
    from oracle import merge as M
    g, p = oracle.default_geometry(n_sectors, tf.max_time_bin), oracle.default_params(cfg.sigma_y_cm, cfg.sigma_z_cm)
    res = oracle.track(g, p, tf.row, tf.pad, tf.time)
    mp = mp if mp is not None else M.default_merge_params(n_sectors)
    mr = M.merge(mp, res.tr_seed, res.tr_sector, res.tr_first_row, res.tr_last_row, res.tr_par)
    mr.refit = oracle.refit_chains(g, p, tf.row, tf.pad, tf.time, res, mr.next, mr.prev)
    return res, mr


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
    # C8: refit of the chains -- flags and counts exact, fits within the stated tolerances (in fact bit-identical)
    ok, ch, cp, rp, rc = (a[go] for a in g["refit"])
    o_ok, o_ch, o_cp, o_rp, o_rc = (a[oo] for a in mr.refit)
    np.testing.assert_array_equal(ok, o_ok, err_msg="refit ok")
    np.testing.assert_array_equal(ch, o_ch, err_msg="chain hits")
    np.testing.assert_array_equal(cp, o_cp, err_msg="chain pieces")
    from parity_util import _check_par
    _check_par(rp, o_rp, "refit")
    assert np.array_equal(rp, o_rp) and np.array_equal(rc, o_rc), "refit not bit-identical"
    assert g["launches_refit"] == 2
    # C9: beam-line time / offset of the refitted states -- one transport each, bit-identical
    from oracle import merge as M
    o_vok, o_vt, o_vy = M.vertex_time(M.default_merge_params(36), o_rp)
    vok, vt, vy = (a[go] for a in g["vertex"])
    np.testing.assert_array_equal(vok, o_vok, err_msg="vertex ok")
    assert np.array_equal(vt, o_vt) and np.array_equal(vy, o_vy), "vertex time / offset not bit-identical"


@pytest.mark.parametrize("seed", [1, 2, 3])
def test_merge_config1_full_tpc(seed):
    cfg = gen.preset(1, seed)
    tf = gen.generate(cfg)
    g = _gpu_track_and_merge(tf, cfg)
    res, mr = _oracle_track_and_merge(tf, cfg)
    _compare(g, res, mr)
    assert mr.n_links > 2000


@pytest.mark.parametrize("cid,seed,us,over", [(2, 1, 150.0, {}), (4, 2, 100.0, {}),
                                              (3, 22091, 120.0, dict(dropout=0.0, noise_frac=0.5))])
def test_merge_continuous_readout_short_frames(cid, seed, us, over):
    """Several overlapping collisions: the time cells of the candidate index and the time_ref differences matter.
    (The third case is the one a randomized sweep found: with this cluster / grid size ratio the arena planner used to put
    the claim array on top of hits_y_time, which the emit kernel reads for the optional hit coordinates.)"""
    cfg = gen.preset(cid, seed, us)
    for k_, v_ in over.items():
        setattr(cfg, k_, v_)
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


def test_full_10ms_frame_merge_invariants_and_sampled_oracle_parity():
    """configs[3] at FULL size, default parameters: tpc_track_timeframe + tpc_merge_tracks as bench.py times them.
    (a) Invariants of the links.  (b) Sampled parity: the oracle tracks and merges the sub-frame {sectors S-2 .. S+2,
    2000-bin window +- 2200 bins}; for every track of sector S whose hits all lie inside the window, the link to its
    continuation (and to the piece it continues) must be the same seed -> seed link as on the GPU (a candidate lies
    within one drift length, 485 bins, of the track, a competitor within another 485: all at least 1200 bins inside
    the sub-frame, where the sampled tracking parity of test_parity_gpu.py holds)."""
    import torch
    from paper_2102_08862_b200 import tracker as T
    from test_parity_gpu import _full_frame, N_ROWS
    import oracle
    from oracle import merge as M
    cfg, tf = _full_frame(3)
    n = tf.n
    trk = T.Tracker(T.default_geometry(36, tf.max_time_bin), T.default_params(cfg.sigma_y_cm, cfg.sigma_z_cm, max_clusters=n))
    d = [torch.from_numpy(a).to(trk.device) for a in (tf.row, tf.pad, tf.time)]
    outs = trk.alloc_outputs(n, hit_coords=True)
    out = trk.tpc_track_timeframe(*d, n=n, outputs=outs)
    nxt, prv, root, n_links = merged = trk.tpc_merge_tracks(outs)
    rf_ok, rf_ch, rf_cp, rf_par, rf_cov = trk.tpc_refit_chains(outs, merged)
    ff = trk.tpc_refit_full(outs, merged)                                        # C12 at full size: sampled parity below
    ce_next, ce_prev, ce_t, ce_n = trk.tpc_merge_central_electrode(outs)        # C10 at full size: invariants below
    torch.cuda.synchronize()
    k, nh = int(out.n_tracks[0]), int(out.n_track_hits[0])
    assert int(out.status[0]) & 7 == 0 and k > 1e6
    ce_next, ce_prev, ce_t, ce_n = ce_next[:k].cpu().numpy(), ce_prev[:k].cpu().numpy(), ce_t[:k].cpu().numpy(), int(ce_n[0])
    dzds_all = out.dzds[:k].cpu().numpy()
    rf_ok, rf_ch, rf_cp, rf_par, rf_cov = (t[:k].cpu().numpy() for t in (rf_ok, rf_ch, rf_cp, rf_par, rf_cov))
    n_hits_all = out.n_hits[:k].cpu().numpy()
    ff_ok, ff_ch, ff_cp, ff_par, ff_cov = (t[:k].cpu().numpy() for t in ff)
    seed, sec = out.seed_hit[:k].cpu().numpy(), out.sector[:k].cpu().numpy()
    first_row, last_row = out.first_row[:k].cpu().numpy(), out.last_row[:k].cpu().numpy()
    x = out.x[:k].cpu().numpy()
    nxt, prv, root, n_links = nxt[:k].cpu().numpy(), prv[:k].cpu().numpy(), root[:k].cpu().numpy(), int(n_links[0])
    trk.close()
    del d, out, outs
    # (a') C10 invariants (as pin CE-I): reciprocal, mirror sectors, approaching the electrode, crossing inside the frame
    ca = np.nonzero(ce_next >= 0)[0]
    cb = ce_next[ca]
    assert ce_n == ca.size and ce_n > 100
    np.testing.assert_array_equal(ce_prev[cb], ca)
    assert np.unique(cb).size == cb.size
    np.testing.assert_array_equal(sec[cb], (sec[ca] + 18) % 36)
    assert np.all(dzds_all[ca] > 0)
    assert np.all(ce_t[ca] > 400.0) and np.all(ce_t[ca] < tf.max_time_bin + 10.0) and np.all(ce_t[ce_next < 0] == 0)
    # (a) invariants (as pin M-I)
    a = np.nonzero(nxt >= 0)[0]
    b = nxt[a]
    assert n_links == a.size and n_links > 2e5
    np.testing.assert_array_equal(prv[b], a)
    assert np.unique(b).size == b.size
    assert np.all(sec[a] // 18 == sec[b] // 18) and np.all(np.isin((sec[a] % 18 - sec[b] % 18) % 18, (1, 17)))
    rb = np.rint((x[b].astype(np.float64) - 85.0) / 1.07).astype(np.int64)
    assert np.all(rb > first_row[a]) and np.all(rb >= last_row[a] - 1) and np.all(rb <= last_row[a] + 13)
    assert np.all(prv[root] == -1) and np.array_equal(root[b], root[a])
    assert k - n_links == np.unique(root).size
    is_root = (prv < 0) & (nxt >= 0)
    assert np.all(rf_ok[~is_root] == 0) and np.all(rf_ok[is_root] != 0) and (rf_ok[is_root] == -1).mean() < 0.03
    np.testing.assert_array_equal(rf_ch[is_root], np.bincount(root, weights=n_hits_all, minlength=k).astype(np.int64)[is_root])
    np.testing.assert_array_equal(rf_cp[is_root], np.bincount(root, minlength=k)[is_root])
    assert np.all(np.isfinite(rf_par)) and np.all(np.isfinite(rf_cov))
    assert np.all(ff_ok[prv >= 0] == 0) and np.all(ff_ok[prv < 0] != 0) and (ff_ok[prv < 0] == -1).mean() < 0.03
    assert np.all(np.isfinite(ff_par)) and np.all(np.isfinite(ff_cov)) and np.all(ff_cov[ff_ok == 1][:, [0, 2, 5, 9, 14]] > 0)
    # (b) sampled parity
    S, t_lo, width, margin = 7, 20000.0, 2000.0, 2200.0
    t_hi = t_lo + width
    sectors = [(S + o) % 18 for o in (-2, -1, 0, 1, 2)]
    srow = (tf.row.astype(np.int64) // N_ROWS)
    sel = np.nonzero(np.isin(srow, sectors) & (tf.time >= t_lo - margin) & (tf.time <= t_hi + margin))[0]
    assert sel.size > 1e6
    o = oracle.track(oracle.default_geometry(36, tf.max_time_bin), oracle.default_params(cfg.sigma_y_cm, cfg.sigma_z_cm),
                     tf.row[sel], tf.pad[sel], tf.time[sel])
    mr = M.merge(M.default_merge_params(36), o.tr_seed, o.tr_sector, o.tr_first_row, o.tr_last_row, o.tr_par)
    o_ok, o_ch, o_cp, o_rp, o_rc = oracle.refit_chains(oracle.default_geometry(36, tf.max_time_bin), oracle.default_params(cfg.sigma_y_cm, cfg.sigma_z_cm),
                                                       tf.row[sel], tf.pad[sel], tf.time[sel], o, mr.next, mr.prev)
    f_ok, f_ch, f_cp, f_rp, f_rc = oracle.refit_full(oracle.default_geometry(36, tf.max_time_bin), oracle.default_params(cfg.sigma_y_cm, cfg.sigma_z_cm),
                                                      tf.row[sel], tf.pad[sel], tf.time[sel], o, mr.next, mr.prev)
    o_t = tf.time[sel][o.tr_hit_index]
    o_min = np.minimum.reduceat(o_t, o.tr_hit_offset); o_max = np.maximum.reduceat(o_t, o.tr_hit_offset)
    core = np.nonzero((o.tr_sector == S) & (o_min >= t_lo) & (o_max <= t_hi))[0]
    assert core.size > 300
    o_seed_global = sel[o.tr_seed]
    lookup = {int(s): i for i, s in enumerate(seed)}
    n_with_link = n_refitted = n_full = 0
    for i in core:
        gi = lookup[int(o_seed_global[i])]                      # the same track exists on the GPU (sampled tracking parity)
        # C8: a chain whose root lies in the core is refitted from the same hits on both sides -> bit-identical
        assert rf_ok[gi] == o_ok[i] and rf_ch[gi] == o_ch[i] and rf_cp[gi] == o_cp[i]
        assert np.array_equal(rf_par[gi], o_rp[i]) and np.array_equal(rf_cov[gi], o_rc[i])
        n_refitted += int(o_ok[i] == 1)
        # C12: every root in the core (single tracks too), full covariance -> bit-identical
        assert ff_ok[gi] == f_ok[i] and ff_ch[gi] == f_ch[i] and ff_cp[gi] == f_cp[i]
        assert np.array_equal(ff_par[gi], f_rp[i]) and np.array_equal(ff_cov[gi], f_rc[i])
        n_full += int(f_ok[i] == 1)
        for o_idx, g_idx in ((mr.next[i], nxt[gi]), (mr.prev[i], prv[gi])):
            o_link = int(o_seed_global[o_idx]) if o_idx >= 0 else -1
            g_link = int(seed[g_idx]) if g_idx >= 0 else -1
            assert o_link == g_link, (int(o_seed_global[i]), o_link, g_link)
            n_with_link += o_link >= 0
    assert n_with_link > 50 and n_refitted > 20 and n_full > 250


def test_refit_with_truncated_hit_lists_flags_the_chains_instead_of_reading_past_the_buffers():
    import torch
    from paper_2102_08862_b200 import tracker as T
    cfg = gen.preset(1, 2)
    tf = gen.generate(cfg)
    n = tf.n
    trk = T.Tracker(T.default_geometry(36, tf.max_time_bin), T.default_params(cfg.sigma_y_cm, cfg.sigma_z_cm, max_clusters=n))
    d = [torch.from_numpy(np.ascontiguousarray(a, np.float32)).to(trk.device) for a in (tf.row, tf.pad, tf.time)]
    outs = trk.alloc_outputs(n, hit_coords=True, max_track_hits=200_000)          # the frame has ~7e5 track hits
    out = trk.tpc_track_timeframe(*d, n=n, outputs=outs)
    merged = trk.tpc_merge_tracks(outs)
    ok, ch, cp, rp, rc = trk.tpc_refit_chains(outs, merged)
    torch.cuda.synchronize()
    k = int(out.n_tracks[0])
    assert int(out.status[0]) & T.STATUS_TRACK_HIT_OVERFLOW and int(out.n_track_hits[0]) > 200_000
    ok, ch = ok[:k].cpu().numpy(), ch[:k].cpu().numpy()
    off, nh = out.hit_offset[:k].cpu().numpy(), out.n_hits[:k].cpu().numpy()
    nxt, prv, root = (t[:k].cpu().numpy() for t in merged[:3])
    roots = np.nonzero((prv < 0) & (nxt >= 0))[0]
    cut = (off + nh) > 200_000                                                      # tracks whose hit list was cut
    chain_cut = np.bincount(root, weights=cut, minlength=k) > 0
    assert np.all(ok[roots[chain_cut[roots]]] == -1) and (ok[roots[~chain_cut[roots]]] == 1).sum() > 100
    assert np.all(np.isfinite(rp[:k].cpu().numpy()))
    trk.close()
