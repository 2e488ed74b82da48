"""GPU parity of C0 (tpc_find_clusters) against oracle/tpc_cluster_oracle.cpp: the peak set is integer work -> exact; the
centres of gravity are one fp32 statement list on both sides -> bit-identical.  And the chain samples -> clusters -> tracks
through both implementations (CUDA cluster finder -> CUDA tracker, oracle cluster finder -> oracle tracker)."""
import numpy as np
import pytest

from paper_2102_08862_b200 import gen
import parity_util as PU

pytestmark = pytest.mark.gpu


def _digits(cid, seed, frame_us=None, **kw):
    c = gen.preset(cid, seed, frame_us)
    for k, v in kw.items():
        setattr(c, k, v)
    tf = gen.generate(c, want_truth=False)
    return c, tf, gen.digitize(tf.row, tf.pad, tf.time, tf.charge, c.n_sectors, tf.max_time_bin)


def _gpu(d, n_sectors, max_time_bin, peak_threshold=8.0, max_clusters=None):
    import torch
    from paper_2102_08862_b200 import tracker as T
    trk = T.Tracker(T.default_geometry(n_sectors, max_time_bin), T.default_params(max_clusters=max(d.n, 1)))
    dev = trk.device
    t = [torch.from_numpy(a).to(dev) for a in (d.row, d.pad, d.time, d.adc)]
    out = trk.tpc_find_clusters(*t, n=d.n, peak_threshold=peak_threshold, max_clusters=max_clusters)
    launches = trk.last_merge_launches()
    torch.cuda.synchronize()
    k = int(out[4][0])
    res = dict(n=k, status=int(out[5][0]), launches=launches, **{nm: out[i][:min(k, out[i].shape[0])].cpu().numpy() for i, nm in enumerate(("row", "pad", "time", "charge"))})
    trk.close()
    return res


def _same(g, o):
    assert g["n"] == o.n and g["status"] == 0
    for nm in ("row", "pad", "time", "charge"):
        assert np.array_equal(g[nm].view(np.uint32), getattr(o, nm).view(np.uint32)), nm


@pytest.mark.parametrize("cid,seed,us", [(0, 1, None), (1, 1, None), (1, 2, None), (2, 1, 200.0), (4, 2, 150.0)])
def test_cluster_finder_matches_the_oracle(cid, seed, us):
    from oracle import clusterfinder as CF
    cfg, tf, d = _digits(cid, seed, us)
    g = _gpu(d, cfg.n_sectors, tf.max_time_bin)
    o = CF.find_clusters(d.row, d.pad, d.time, d.adc)
    _same(g, o)
    assert o.n > 0.8 * tf.n and g["launches"] == 5


def test_cluster_finder_other_threshold_ties_and_degenerate_inputs():
    from oracle import clusterfinder as CF
    cfg, tf, d = _digits(0, 5)
    for thr in (3.0, 25.0, 1000.0):
        _same(_gpu(d, 1, tf.max_time_bin, peak_threshold=thr), CF.find_clusters(d.row, d.pad, d.time, d.adc, thr))
    # plateaus: every ADC the same -> ties everywhere, decided on the input order
    flat = gen.Digits(d.row, d.pad, d.time, np.full(d.n, 20.0, np.float32))
    _same(_gpu(flat, 1, tf.max_time_bin), CF.find_clusters(flat.row, flat.pad, flat.time, flat.adc))
    # long groups (a whole pad row lit in one time bin) and isolated samples
    row = np.concatenate([np.full(120, 5), np.full(120, 5), [7, 9]]).astype(np.int32)
    pad = np.concatenate([np.arange(120), np.arange(120), [3, 3]]).astype(np.int32)
    time = np.concatenate([np.full(120, 40), np.full(120, 41), [40, 40]]).astype(np.int32)
    adc = (10 + (np.arange(242) * 7919) % 23).astype(np.float32)
    dd = gen.Digits(row, pad, time, adc)
    _same(_gpu(dd, 1, 487.0), CF.find_clusters(row, pad, time, adc))
    e = gen.Digits(*(np.zeros(0, np.int32) for _ in range(3)), np.zeros(0, np.float32))
    assert _gpu(e, 1, 487.0)["n"] == 0
    # capacity: more clusters than max_clusters -> status 1, count reported, a valid prefix written
    full = _gpu(d, 1, tf.max_time_bin)
    cut = _gpu(d, 1, tf.max_time_bin, max_clusters=100)
    assert cut["status"] == 1 and cut["n"] == full["n"] and np.array_equal(cut["pad"][:100], full["pad"][:100])


def test_cluster_finder_groups_longer_than_the_staged_halo_take_the_global_memory_window():
    """A (sector_row, time bin) with more samples than half the halo of a tile (352 samples) cannot be staged completely for
    every tile that touches it: those samples are served by cf_window_global.  Wide groups across several tile boundaries
    (tile = 2048 samples), with plateaus so that the tie rule is exercised there too."""
    from oracle import clusterfinder as CF
    rng = np.random.default_rng(12)
    rows, pads, times, adcs = [], [], [], []
    for t in range(1700):                                              # filler: isolated samples of row 0, one per time bin
        rows.append([0]); pads.append([t % 60]); times.append([2 * t]); adcs.append([30.0])
    for r, width in ((1, 500), (2, 900), (3, 353), (4, 352)):          # then four rows with wide groups in 6 consecutive time bins
        for t in range(100, 106):
            lit = np.sort(rng.choice(1000, width, replace=False))
            rows.append(np.full(width, r)); pads.append(lit); times.append(np.full(width, t))
            adcs.append(rng.integers(5, 12, width).astype(np.float32) * 4.0)
    for t in range(900):
        rows.append([5]); pads.append([7]); times.append([3 * t]); adcs.append([9.0])
    row, pad, time = (np.concatenate(v).astype(np.int32) for v in (rows, pads, times))
    adc = np.concatenate(adcs).astype(np.float32)
    assert row.size > 6 * 2048
    dd = gen.Digits(row, pad, time, adc)
    o = CF.find_clusters(row, pad, time, adc)
    g = _gpu(dd, 1, 4000.0)
    _same(g, o)
    assert o.n > 3000


def test_cluster_finder_survives_unsorted_and_duplicated_input():
    """The contract wants sorted, duplicate-free samples; anything else gives unspecified clusters but must not fault."""
    import torch
    rng = np.random.default_rng(3)
    n = 50_000
    dd = gen.Digits(rng.integers(-3, 200, n).astype(np.int32), rng.integers(-5, 140, n).astype(np.int32),
                    rng.integers(-2, 500, n).astype(np.int32), rng.uniform(0, 60, n).astype(np.float32))
    g = _gpu(dd, 1, 487.0)
    assert 0 <= g["n"] <= n
    same = gen.Digits(np.full(n, 3, np.int32), np.full(n, 9, np.int32), np.full(n, 17, np.int32), np.full(n, 20.0, np.float32))
    g = _gpu(same, 1, 487.0)                                           # one group of 50 000 duplicates
    assert 0 <= g["n"] <= n
    torch.cuda.synchronize()


def test_samples_to_tracks_through_both_implementations():
    """samples -> clusters -> tracks: CUDA cluster finder + CUDA tracker against oracle cluster finder + oracle tracker."""
    from oracle import clusterfinder as CF
    cfg, tf, d = _digits(1, 3)
    g = _gpu(d, 36, tf.max_time_bin)
    o = CF.find_clusters(d.row, d.pad, d.time, d.adc)
    _same(g, o)
    gt = PU.run_gpu(g["row"], g["pad"], g["time"], 36, tf.max_time_bin)
    ot = PU.run_oracle(o.row, o.pad, o.time, 36, tf.max_time_bin)
    rep = PU.compare(gt, ot)
    assert rep["n_tracks"] > 5000 and rep["track_par_bit_identical"]
