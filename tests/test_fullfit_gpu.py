"""GPU parity of C12 (tpc_refit_full: Kalman refit with the full 5x5 covariance, multiple scattering and energy loss)
against oracle/tpc_oracle.cpp::orc_refit_full.  Both sides fit THEIR OWN tracks and links (CUDA tracker -> CUDA merger ->
CUDA refit, oracle likewise); tracks are joined on their seed id.  Flags and counts are integer work (exact); the fits are
fp32 in the same operation order and come out bit-identical, which is what is asserted.  The full 10 ms frame is covered by
tests/test_merge_gpu.py::test_full_10ms_frame_merge_invariants_and_sampled_oracle_parity.
"""
from __future__ import annotations

import numpy as np
import pytest

from paper_2102_08862_b200 import gen

pytestmark = pytest.mark.gpu

GAS = (1.0 / 3.0e4, 1.7e-6, 0.13957, 0.1)
DENSE = (1.0 / 300.0, 1.7e-5, 0.13957, 0.3)           # a hundred times the scattering, ten times the stopping power
KAON_NO_STRAGGLING = (1.0 / 3.0e4, 1.7e-6, 0.49368, 0.0)
NONE = (0.0, 0.0, 0.13957, 0.0)


def _gpu(tf, cfg, materials, max_track_hits=None):
    import torch
    from paper_2102_08862_b200 import tracker as T
    n = tf.n
    trk = T.Tracker(T.default_geometry(36, tf.max_time_bin), T.default_params(cfg.sigma_y_cm, cfg.sigma_z_cm, max_clusters=max(n, 1)))
    d = [torch.from_numpy(np.ascontiguousarray(a, np.float32)).to(trk.device) for a in (tf.row, tf.pad, tf.time)]
    outs = trk.alloc_outputs(n, hit_coords=True) if max_track_hits is None else trk.alloc_outputs(n, hit_coords=True, max_track_hits=max_track_hits)
    out = trk.tpc_track_timeframe(*d, n=n, outputs=outs)
    merged = trk.tpc_merge_tracks(outs)
    fits = []
    for m in materials:
        fits.append(trk.tpc_refit_full(outs, merged, m))
        assert trk.last_merge_launches() == 2
    torch.cuda.synchronize()
    k = int(out.n_tracks[0])
    g = dict(k=k, status=int(out.status[0]), seed=out.seed_hit[:k].cpu().numpy(), fits=[tuple(t[:k].cpu().numpy() for t in f) for f in fits],
             next=merged[0][:k].cpu().numpy(), prev=merged[1][:k].cpu().numpy(), root=merged[2][:k].cpu().numpy(),
             off=out.hit_offset[:k].cpu().numpy(), nh=out.n_hits[:k].cpu().numpy(), n_track_hits=int(out.n_track_hits[0]))
    trk.close()
    return g


def _oracle(tf, cfg, materials):
    import oracle
    from oracle import merge as M
    g, p = oracle.default_geometry(36, tf.max_time_bin), oracle.default_params(cfg.sigma_y_cm, cfg.sigma_z_cm)
    res = oracle.track(g, p, tf.row, tf.pad, tf.time)
    mr = M.merge(M.default_merge_params(36), res.tr_seed, res.tr_sector, res.tr_first_row, res.tr_last_row, res.tr_par)
    return res, mr, [oracle.refit_full(g, p, tf.row, tf.pad, tf.time, res, mr.next, mr.prev, m) for m in materials]


def _compare(g, res, mr, o_fits):
    assert g["status"] & 7 == 0 and g["k"] == len(res.tr_seed)
    go, oo = np.argsort(g["seed"], kind="stable"), np.argsort(res.tr_seed, kind="stable")
    np.testing.assert_array_equal(g["seed"][go], res.tr_seed[oo])
    for fit, o_fit in zip(g["fits"], o_fits):
        ok, ch, cp, rp, rc = (a[go] for a in fit)
        o_ok, o_ch, o_cp, o_rp, o_rc = (a[oo] for a in o_fit)
        np.testing.assert_array_equal(ok, o_ok, err_msg="ok")
        np.testing.assert_array_equal(ch, o_ch, err_msg="chain hits")
        np.testing.assert_array_equal(cp, o_cp, err_msg="chain pieces")
        bad = np.nonzero(np.any(rp != o_rp, axis=1) | np.any(rc != o_rc, axis=1))[0]
        assert bad.size == 0, (bad.size, rp[bad[:3]], o_rp[bad[:3]], rc[bad[:3]], o_rc[bad[:3]])
        assert (ok == 1).sum() > 0.9 * (mr.prev < 0).sum()


@pytest.mark.parametrize("seed", [1, 2])
def test_fullfit_config1_full_tpc_four_materials(seed):
    cfg = gen.preset(1, seed)
    tf = gen.generate(cfg)
    mats = [GAS, DENSE, KAON_NO_STRAGGLING, NONE]
    g = _gpu(tf, cfg, mats)
    res, mr, o_fits = _oracle(tf, cfg, mats)
    _compare(g, res, mr, o_fits)
    # the materials really differ in the result, and chains of three pieces are among the fitted roots
    assert not np.array_equal(g["fits"][0][3], g["fits"][1][3]) and not np.array_equal(g["fits"][0][3], g["fits"][2][3])
    assert not np.array_equal(g["fits"][0][4], g["fits"][3][4])
    assert (g["fits"][0][2][g["fits"][0][0] == 1] >= 3).sum() > 50


@pytest.mark.parametrize("cid,seed,us", [(0, 3, None), (2, 1, 150.0), (3, 7, 120.0), (4, 2, 100.0)])
def test_fullfit_other_configs(cid, seed, us):
    cfg = gen.preset(cid, seed) if us is None else gen.preset(cid, seed, us)
    tf = gen.generate(cfg)
    g = _gpu(tf, cfg, [GAS])
    res, mr, o_fits = _oracle(tf, cfg, [GAS])
    _compare(g, res, mr, o_fits)


def test_fullfit_with_truncated_hit_lists_flags_the_roots_instead_of_reading_past_the_buffers():
    cfg = gen.preset(1, 2)
    tf = gen.generate(cfg)
    import torch
    from paper_2102_08862_b200 import tracker as T
    n = tf.n
    trk = T.Tracker(T.default_geometry(36, tf.max_time_bin), T.default_params(cfg.sigma_y_cm, cfg.sigma_z_cm, max_clusters=n))
    d = [torch.from_numpy(np.ascontiguousarray(a, np.float32)).to(trk.device) for a in (tf.row, tf.pad, tf.time)]
    outs = trk.alloc_outputs(n, hit_coords=True, max_track_hits=200_000)      # the frame has ~7e5 track hits
    out = trk.tpc_track_timeframe(*d, n=n, outputs=outs)
    merged = trk.tpc_merge_tracks(outs)
    ok, ch, cp, rp, rc = trk.tpc_refit_full(outs, merged)
    torch.cuda.synchronize()
    k = int(out.n_tracks[0])
    assert int(out.status[0]) & T.STATUS_TRACK_HIT_OVERFLOW and int(out.n_track_hits[0]) > 200_000
    ok = ok[:k].cpu().numpy()
    off, nh = out.hit_offset[:k].cpu().numpy(), out.n_hits[:k].cpu().numpy()
    nxt, prv, root = (t[:k].cpu().numpy() for t in merged[:3])
    roots = np.nonzero(prv < 0)[0]
    cut = (off + nh) > 200_000                                                  # tracks whose hit list was cut
    chain_cut = np.bincount(root, weights=cut, minlength=k) > 0
    assert np.all(ok[roots[chain_cut[roots]]] == -1) and (ok[roots[~chain_cut[roots]]] == 1).sum() > 1000
    assert np.all(np.isfinite(rp[:k].cpu().numpy())) and np.all(np.isfinite(rc[:k].cpu().numpy()))
    trk.close()


def test_fullfit_rejects_bad_arguments():
    import torch
    from paper_2102_08862_b200 import tracker as T
    cfg = gen.preset(0, 1)
    tf = gen.generate(cfg)
    n = tf.n
    trk = T.Tracker(T.default_geometry(36, tf.max_time_bin), T.default_params(cfg.sigma_y_cm, cfg.sigma_z_cm, max_clusters=n))
    d = [torch.from_numpy(np.ascontiguousarray(a, np.float32)).to(trk.device) for a in (tf.row, tf.pad, tf.time)]
    outs = trk.alloc_outputs(n, hit_coords=True)
    trk.tpc_track_timeframe(*d, n=n, outputs=outs)
    merged = trk.tpc_merge_tracks(outs)
    for bad in [(-1.0, 1e-6, 0.1, 0.1), (1e-4, -1e-6, 0.1, 0.1), (1e-4, 1e-6, -0.1, 0.1), (1e-4, 1e-6, 0.1, float("nan"))]:
        with pytest.raises(T.TpcError):
            trk.tpc_refit_full(outs, merged, bad)
    no_coords = trk.alloc_outputs(n, hit_coords=False)
    trk.tpc_track_timeframe(*d, n=n, outputs=no_coords)
    with pytest.raises(T.TpcError):
        trk.tpc_refit_full(no_coords, trk.tpc_merge_tracks(no_coords))
    torch.cuda.synchronize()
    trk.close()


def _gpu_ce(tf, cfg, material):
    import torch
    from paper_2102_08862_b200 import tracker as T
    n = tf.n
    trk = T.Tracker(T.default_geometry(36, tf.max_time_bin), T.default_params(max(cfg.sigma_y_cm, 0.08), max(cfg.sigma_z_cm, 0.12), max_clusters=max(n, 1)))
    d = [torch.from_numpy(np.ascontiguousarray(a, np.float32)).to(trk.device) for a in (tf.row, tf.pad, tf.time)]
    outs = trk.alloc_outputs(n, hit_coords=True)
    out = trk.tpc_track_timeframe(*d, n=n, outputs=outs)
    merged = trk.tpc_merge_tracks(outs)
    ce = trk.tpc_merge_central_electrode(outs)
    fit = trk.tpc_refit_full(outs, merged, material, ce_merged=ce)
    plain = trk.tpc_refit_full(outs, merged, material)
    torch.cuda.synchronize()
    k = int(out.n_tracks[0])
    g = dict(k=k, status=int(out.status[0]), seed=out.seed_hit[:k].cpu().numpy(), fits=[tuple(t[:k].cpu().numpy() for t in f) for f in (fit, plain)],
             ce_links=int(ce[3][0]))
    trk.close()
    return g


@pytest.mark.parametrize("seed,noise_free", [(3, True), (4, False), (5, False)])
def test_fullfit_across_the_central_electrode(seed, noise_free):
    import oracle
    from oracle import merge as M
    cfg = gen.preset(1, seed)
    cfg.fixed_tracks, cfg.zv_sigma_cm, cfg.eta_max, cfg.pt_min = 3000, 30.0, 0.3, 0.3        # many tracks through the electrode INSIDE the TPC
    if noise_free:
        cfg.sigma_y_cm = cfg.sigma_z_cm = cfg.dropout = cfg.noise_frac = 0.0
    tf = gen.generate(cfg, want_truth=False)
    g = _gpu_ce(tf, cfg, GAS)
    geo, par = oracle.default_geometry(36, tf.max_time_bin), oracle.default_params(max(cfg.sigma_y_cm, 0.08), max(cfg.sigma_z_cm, 0.12))
    res = oracle.track(geo, par, tf.row, tf.pad, tf.time)
    mr = M.merge(M.default_merge_params(36), res.tr_seed, res.tr_sector, res.tr_first_row, res.tr_last_row, res.tr_par)
    ce = M.merge_ce(M.default_ce_params(36), res.tr_seed, res.tr_sector, res.tr_first_row, res.tr_last_row, res.tr_par)
    o_fit = oracle.refit_full_ce(geo, par, tf.row, tf.pad, tf.time, res, mr.next, mr.prev, ce.next, ce.prev, ce.t_ce, GAS)
    o_plain = oracle.refit_full(geo, par, tf.row, tf.pad, tf.time, res, mr.next, mr.prev, GAS)
    assert g["ce_links"] == ce.n_links >= 150
    _compare(g, res, mr, [o_fit, o_plain])
    # the electrode really is crossed by fitted chains: roots whose chain is longer than without C10's links
    longer = (o_fit[1] > o_plain[1]) & (o_fit[0] == 1)
    assert longer.sum() >= 0.9 * ce.n_links and (o_fit[0] == 0).sum() > (o_plain[0] == 0).sum()
