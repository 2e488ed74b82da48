"""GPU parity of C10 (tpc_merge_central_electrode) against oracle/tpc_merge_oracle.cpp::orc_merge_ce: links are integer
work -> bit-exact; the crossing time is one fp32 statement list on both sides -> bit-identical.

Both sides get THEIR OWN tracks (CUDA tracker -> CUDA merger, oracle tracker -> oracle merger); tracks are joined on the
seed.  The frames are the generator's with a wide vertex spread and flat tracks, so that hundreds of them pass the central
electrode INSIDE the TPC volume (with the default 5 cm vertex spread most crossings happen below the first pad row).
"""
import numpy as np
import pytest

from paper_2102_08862_b200 import gen

pytestmark = pytest.mark.gpu


def _frame(cid, seed, frame_us=None, wide=True, **kw):
    c = gen.preset(cid, seed, frame_us)
    if wide:
        c.zv_sigma_cm, c.eta_max, c.pt_min = 30.0, 0.3, 0.3
    for k, v in kw.items():
        setattr(c, k, v)
    return c, gen.generate(c, want_truth=False)


def _gpu(tf, cfg, ce_params=None, n_sectors=36):
    import torch
    from paper_2102_08862_b200 import tracker as T
    n = tf.n
    trk = T.Tracker(T.default_geometry(n_sectors, tf.max_time_bin), T.default_params(max(cfg.sigma_y_cm, 0.08), max(cfg.sigma_z_cm, 0.12), max_clusters=max(n, 1)))
    d = [torch.from_numpy(np.ascontiguousarray(a, np.float32)).to(trk.device) for a in (tf.row, tf.pad, tf.time)]
    outs = trk.alloc_outputs(n)
    out = trk.tpc_track_timeframe(*d, n=n, outputs=outs)
    mg = trk.tpc_merge_tracks(outs)                        # C7 first: C10 reuses (overwrites) its scratch
    nxt, prv, tce, nl = trk.tpc_merge_central_electrode(outs, ce_params)
    launches = trk.last_merge_launches()
    work = trk.work_counters()                             # the counter block survives the merge calls (it is not in the arena)
    torch.cuda.synchronize()
    k = int(out.n_tracks[0])
    res = dict(k=k, seed=out.seed_hit[:k].cpu().numpy(), next=nxt.cpu().numpy(), prev=prv.cpu().numpy(), t_ce=tce.cpu().numpy(),
               n_links=int(nl[0]), launches=launches, status=int(out.status[0]), c7_links=int(mg[3][0]), work=work)
    trk.close()
    return res


def _oracle(tf, cfg, ce=None, n_sectors=36):
    import oracle
    from oracle import merge as M
    res = oracle.track(oracle.default_geometry(n_sectors, tf.max_time_bin), oracle.default_params(max(cfg.sigma_y_cm, 0.08), max(cfg.sigma_z_cm, 0.12)),
                       tf.row, tf.pad, tf.time)
    ce = ce if ce is not None else M.default_ce_params(n_sectors)
    return res, M.merge_ce(ce, res.tr_seed, res.tr_sector, res.tr_first_row, res.tr_last_row, res.tr_par)


def _links(seed, idx):
    return np.where(idx >= 0, seed[np.maximum(idx, 0)], -1)


def _compare(g, res, r):
    k = g["k"]
    assert g["status"] & 7 == 0 and k == len(res.tr_seed)
    go, oo = np.argsort(g["seed"], kind="stable"), np.argsort(res.tr_seed, kind="stable")
    np.testing.assert_array_equal(g["seed"][go], res.tr_seed[oo])
    np.testing.assert_array_equal(_links(g["seed"], g["next"][:k])[go], _links(res.tr_seed, r.next)[oo], err_msg="next")
    np.testing.assert_array_equal(_links(g["seed"], g["prev"][:k])[go], _links(res.tr_seed, r.prev)[oo], err_msg="prev")
    assert np.array_equal(g["t_ce"][:k][go].view(np.uint32), r.t_ce[oo].view(np.uint32)), "crossing times not bit-identical"
    assert g["n_links"] == r.n_links
    assert np.all(g["next"][k:] == -1) and np.all(g["prev"][k:] == -1) and np.all(g["t_ce"][k:] == 0)
    assert g["launches"] >= 7


@pytest.mark.parametrize("seed,noise_free", [(3, True), (4, False), (5, False)])
def test_ce_merge_frames_with_many_crossings(seed, noise_free):
    kw = dict(sigma_y_cm=0.0, sigma_z_cm=0.0, dropout=0.0, noise_frac=0.0) if noise_free else {}
    cfg, tf = _frame(1, seed, fixed_tracks=3000, **kw)
    g = _gpu(tf, cfg)
    res, r = _oracle(tf, cfg)
    _compare(g, res, r)
    assert r.n_links >= 150
    assert g["work"]["tracklets"] > 1000                    # tpc_tracker_work_counters is still valid after two merge calls


@pytest.mark.parametrize("cid,seed,us", [(1, 1, None), (2, 1, 150.0), (3, 2, 200.0), (4, 1, 120.0)])
def test_ce_merge_baseline_configs(cid, seed, us):
    """The BASELINE.json generator as it is (5 cm vertex spread: few crossings inside the TPC, many loopers)."""
    cfg, tf = _frame(cid, seed, us, wide=False)
    g = _gpu(tf, cfg)
    res, r = _oracle(tf, cfg)
    _compare(g, res, r)


def test_ce_merge_other_cuts():
    from paper_2102_08862_b200 import tracker as T
    from oracle import merge as M
    cfg, tf = _frame(1, 6, fixed_tracks=2500)
    g = _gpu(tf, cfg, ce_params=T.CeParams(0.8, 4.0, 0.02, 0.3, 0.04, 5, 0))
    ce = M.default_ce_params(36)
    ce.cut_y_cm, ce.cut_z_cm, ce.cut_sin_phi, ce.cut_q_pt, ce.cut_dzds, ce.max_row_gap, ce.max_row_overlap = 0.8, 4.0, 0.02, 0.3, 0.04, 5, 0
    res, r = _oracle(tf, cfg, ce=ce)
    _compare(g, res, r)
    assert 20 <= r.n_links


def test_ce_merge_half_tpc_empty_frame_and_bad_arguments():
    import torch
    from paper_2102_08862_b200 import tracker as T
    cfg, tf = _frame(0, 1, wide=False)
    g = _gpu(tf, cfg, n_sectors=1)
    assert g["n_links"] == 0 and np.all(g["next"] == -1) and np.all(g["t_ce"] == 0)
    trk = T.Tracker(T.default_geometry(36, 487.0), T.default_params(max_clusters=1000))
    e = torch.zeros(0, dtype=torch.float32, device=trk.device)
    outs = trk.alloc_outputs(0)
    trk.tpc_track_timeframe(e, e, e, n=0, outputs=outs)
    nxt, prv, tce, nl = trk.tpc_merge_central_electrode(outs)
    torch.cuda.synchronize()
    assert int(nl[0]) == 0
    with pytest.raises(T.TpcError):
        trk.tpc_merge_central_electrode(outs, T.CeParams(2.0, 2.0, 0.05, 0.5, 0.0, 12, 2))
    trk.close()
