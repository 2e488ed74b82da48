"""GPU parity of C11 (tpc_compress_tracks) against oracle::orc_compress_tracks: rejection flags and symbols are integers ->
bit-exact.  Both sides get THEIR OWN tracks (CUDA tracker -> CUDA coder, oracle tracker -> oracle coder); tracks joined on
the seed, hits compared in hit_index order (identical on both sides by the tracking parity)."""
import numpy as np
import pytest

from paper_2102_08862_b200 import gen

pytestmark = pytest.mark.gpu


def _frame(cid, seed, frame_us=None, **kw):
    c = gen.preset(cid, seed, frame_us)
    for k, v in kw.items():
        setattr(c, k, v)
    return c, gen.generate(c, want_truth=False)


def _gpu(tf, cfg, **ckw):
    import torch
    from paper_2102_08862_b200 import tracker as T
    n = tf.n
    trk = T.Tracker(T.default_geometry(cfg.n_sectors, tf.max_time_bin), T.default_params(cfg.sigma_y_cm, cfg.sigma_z_cm, max_clusters=max(n, 1)))
    d = [torch.from_numpy(np.ascontiguousarray(a, np.float32)).to(trk.device) for a in (tf.row, tf.pad, tf.time)]
    outs = trk.alloc_outputs(n, hit_coords=True)
    out = trk.tpc_track_timeframe(*d, n=n, outputs=outs)
    rej, ok, qy, qz = trk.tpc_compress_tracks(outs, n, **ckw)
    launches = trk.last_merge_launches()
    torch.cuda.synchronize()
    k, nh = int(out.n_tracks[0]), int(out.n_track_hits[0])
    res = dict(k=k, nh=nh, seed=out.seed_hit[:k].cpu().numpy(), n_hits=out.n_hits[:k].cpu().numpy(), off=out.hit_offset[:k].cpu().numpy(),
               hit_index=out.hit_index[:nh].cpu().numpy(), reject=rej[:n].cpu().numpy(), ok=ok[:k].cpu().numpy(), qy=qy[:nh].cpu().numpy(),
               qz=qz[:nh].cpu().numpy(), launches=launches, status=int(out.status[0]))
    trk.close()
    return res


def _oracle(tf, cfg, **ckw):
    import oracle
    g, p = oracle.default_geometry(cfg.n_sectors, tf.max_time_bin), oracle.default_params(cfg.sigma_y_cm, cfg.sigma_z_cm)
    res = oracle.track(g, p, tf.row, tf.pad, tf.time)
    kw = {{"reject_q_pt": "reject_qpt"}.get(k, k): v for k, v in ckw.items()}
    return res, oracle.compress_tracks(g, p, tf.row, tf.pad, tf.time, res, **kw)


def _compare(g, res, c):
    import parity_util as PU
    rej, ok, qy, qz = c
    assert g["status"] & 7 == 0 and g["k"] == len(res.tr_seed) and g["nh"] == len(res.tr_hit_index)
    np.testing.assert_array_equal(g["reject"], rej, err_msg="reject flags")
    go, oo = np.argsort(g["seed"], kind="stable"), np.argsort(res.tr_seed, kind="stable")
    np.testing.assert_array_equal(g["seed"][go], res.tr_seed[oo])
    np.testing.assert_array_equal(g["ok"][go], ok[oo], err_msg="ok")
    np.testing.assert_array_equal(g["n_hits"][go], res.tr_n_hits[oo])
    for a, b, nm in ((g["qy"], qy, "res_y"), (g["qz"], qz, "res_z"), (g["hit_index"], res.tr_hit_index, "hit_index")):
        np.testing.assert_array_equal(PU._ragged_gather(a, g["off"][go], g["n_hits"][go]), PU._ragged_gather(b, res.tr_hit_offset[oo], res.tr_n_hits[oo]), err_msg=nm)
    assert g["launches"] == 2


@pytest.mark.parametrize("cid,seed,us", [(0, 1, None), (1, 1, None), (1, 3, None), (2, 1, 150.0), (4, 2, 150.0)])
def test_compress_matches_the_oracle(cid, seed, us):
    cfg, tf = _frame(cid, seed, us)
    g = _gpu(tf, cfg)
    res, c = _oracle(tf, cfg)
    _compare(g, res, c)
    assert (c[1] == 1).sum() > 50 and (cid == 0 or (c[1] == -1).sum() >= 1)


def test_compress_other_parameters_and_low_momentum_tracks():
    cfg, tf = _frame(1, 2, pt_min=0.05)                        # loopers: many rejected tracks, some transport FAILs while coding
    for kw in (dict(reject_q_pt=1.0 / 0.2, step_y=0.01, step_z=0.05), dict(reject_q_pt=1e9, step_y=0.2, step_z=0.2), dict(reject_q_pt=0.5)):
        g = _gpu(tf, cfg, **kw)
        res, c = _oracle(tf, cfg, **kw)
        _compare(g, res, c)
    assert (c[1] == -1).sum() > 0.5 * len(c[1])                # the last cut rejects most tracks


def test_compress_empty_frame_and_bad_arguments():
    import torch
    from paper_2102_08862_b200 import tracker as T
    trk = T.Tracker(T.default_geometry(36, 487.0), T.default_params(max_clusters=1000))
    e = torch.zeros(0, dtype=torch.float32, device=trk.device)
    outs = trk.alloc_outputs(0, hit_coords=True)
    trk.tpc_track_timeframe(e, e, e, n=0, outputs=outs)
    rej, ok, qy, qz = trk.tpc_compress_tracks(outs, 0)
    torch.cuda.synchronize()
    with pytest.raises(T.TpcError):
        trk.tpc_compress_tracks(outs, 0, step_y=0.0)
    no_coords = trk.alloc_outputs(10)
    with pytest.raises(T.TpcError):
        trk.tpc_compress_tracks(no_coords, 10)
    trk.close()
