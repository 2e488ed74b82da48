"""Pins of the C0 oracle (oracle/tpc_cluster_oracle.cpp: the TPC cluster finder).

The paper names the step and prints nothing about it, so the pins are what the definition and the
generator fix: D-C the centre of gravity against its closed form, D-B a dense-array restatement on small frames, D-T the
tie rule, D-I invariants, D-E clusters -> samples -> clusters recovers isolated clusters, D-O the input contract.
"""
import numpy as np
import pytest

from oracle import clusterfinder as CF
from paper_2102_08862_b200 import gen


def _sorted(row, pad, time, adc):
    row, pad, time = (np.asarray(a, np.int32) for a in (row, pad, time))
    adc = np.asarray(adc, np.float32)
    o = np.lexsort((pad, time, row))
    return row[o], pad[o], time[o], adc[o]


def test_DC_centre_of_gravity_of_one_deposit_is_the_closed_form():
    a = np.array([[3, 9, 4], [12, 40, 17], [5, 11, 6]], np.float32)          # [time offset][pad offset]
    row, pad, time, adc = [], [], [], []
    for it in range(3):
        for ip in range(3):
            row.append(7); pad.append(50 + ip); time.append(200 + it); adc.append(a[it, ip])
    c = CF.find_clusters(*_sorted(row, pad, time, adc))
    assert c.n == 1 and c.row[0] == 7.0 and c.charge[0] == a.sum()
    q = float(a.sum())
    assert abs(float(c.pad[0]) - (51 + float((a * np.array([-1, 0, 1])[None, :]).sum()) / q)) < 1e-5
    assert abs(float(c.time[0]) - (201 + float((a * np.array([-1, 0, 1])[:, None]).sum()) / q)) < 1e-5
    # below the peak threshold: nothing; exactly at it: a cluster
    lo = a * np.float32(7.0 / 40.0)
    assert CF.find_clusters(*_sorted(row, pad, time, lo.reshape(-1)), peak_threshold=8.0).n == 0
    assert CF.find_clusters(*_sorted(row, pad, time, (a / 5).reshape(-1)), peak_threshold=8.0).n == 1
    # samples of another sector-row, two pads away or two time bins away do not enter
    row2 = row + [8, 7, 7]; pad2 = pad + [51, 53, 51]; time2 = time + [201, 201, 203]; adc2 = list(a.reshape(-1)) + [30, 30, 30]
    c2 = CF.find_clusters(*_sorted(row2, pad2, time2, adc2))
    i = int(np.argmax(c2.charge == a.sum()))
    assert c2.n == 4 and c2.pad[i] == c.pad[0] and c2.time[i] == c.time[0]


def _dense_restatement(row, pad, time, adc, thr):
    """The definition again on a dense [time][pad] array per sector-row, fp32 sums in the stated order."""
    f = np.float32
    out = []
    index = {(int(r), int(p), int(t)): i for i, (r, p, t) in enumerate(zip(row, pad, time))}
    for r in np.unique(row):
        m = row == r
        T, P = int(time[m].max()) + 3, int(pad[m].max()) + 3
        grid = np.full((T, P), -1.0, np.float32)                  # -1 = no sample
        grid[time[m] + 1, pad[m] + 1] = adc[m]
        for t, p in zip(time[m], pad[m]):
            a0 = grid[t + 1, p + 1]
            if not a0 >= thr:
                continue
            me = index[(int(r), int(p), int(t))]
            ok, q, sp, st = True, f(0), f(0), f(0)
            for dt in (-1, 0, 1):
                for dp in (-1, 0, 1):
                    a = grid[t + 1 + dt, p + 1 + dp]
                    if a < 0:
                        continue
                    if (dt, dp) != (0, 0):
                        e = index[(int(r), int(p + dp), int(t + dt))]
                        if not (a0 > a or (a0 == a and me < e)):
                            ok = False
                    q = f(q + a); sp = f(sp + f(dp) * a); st = f(st + f(dt) * a)
            if ok:
                out.append((me, f(p) + f(sp / q), f(t) + f(st / q), q))
    out.sort()
    return out


@pytest.mark.parametrize("seed", [1, 2])
def test_DB_dense_array_restatement_on_a_small_frame(seed):
    c = gen.preset(0, seed)
    c.fixed_tracks = 25
    tf = gen.generate(c)
    d = gen.digitize(tf.row, tf.pad, tf.time, tf.charge, 1, tf.max_time_bin)
    assert 3000 < d.n < 30000
    got = CF.find_clusters(d.row, d.pad, d.time, d.adc, 8.0)
    ref = _dense_restatement(d.row, d.pad, d.time, d.adc, np.float32(8.0))
    assert got.n == len(ref) > 500
    np.testing.assert_array_equal(got.peak, [x[0] for x in ref])
    assert np.array_equal(got.pad, np.array([x[1] for x in ref], np.float32))
    assert np.array_equal(got.time, np.array([x[2] for x in ref], np.float32))
    assert np.array_equal(got.charge, np.array([x[3] for x in ref], np.float32))


def test_DT_ties_go_to_the_earlier_sample():
    # a 2 x 2 plateau: exactly one peak, the first in (time, pad) order, whose 3 x 3 window holds all four samples
    row, pad, time, adc = _sorted([3] * 4, [10, 11, 10, 11], [100, 100, 101, 101], [20, 20, 20, 20])
    c = CF.find_clusters(row, pad, time, adc)
    assert c.n == 1 and c.peak[0] == 0 and c.charge[0] == 80.0 and c.pad[0] == 10.5 and c.time[0] == 100.5
    # two equal samples three pads apart are two clusters; two pads apart with an equal one in between: the first wins, the
    # third is not a neighbour of the first and is beaten by the second -> one cluster
    c = CF.find_clusters(*_sorted([3, 3], [10, 13], [100, 100], [20, 20]))
    assert c.n == 2
    c = CF.find_clusters(*_sorted([3, 3, 3], [10, 11, 12], [100, 100, 100], [20, 20, 20]))
    assert c.n == 1 and c.peak[0] == 0 and c.charge[0] == 40.0


def test_DO_input_contract():
    with pytest.raises(ValueError):
        CF.find_clusters([3, 3], [11, 10], [100, 100], [20.0, 20.0])          # pads not ascending
    with pytest.raises(ValueError):
        CF.find_clusters([3, 3], [10, 10], [100, 100], [20.0, 20.0])          # duplicate
    assert CF.find_clusters([], [], [], []).n == 0


@pytest.mark.parametrize("cid,seed", [(0, 3), (1, 2)])
def test_DI_invariants_and_DE_generated_clusters_are_recovered(cid, seed):
    cfg = gen.preset(cid, seed)
    tf = gen.generate(cfg)
    d = gen.digitize(tf.row, tf.pad, tf.time, tf.charge, cfg.n_sectors, tf.max_time_bin)
    c = CF.find_clusters(d.row, d.pad, d.time, d.adc)
    # D-I: a peak is at least the threshold, the centroid stays within one cell of it, no two peaks are neighbours
    assert np.all(d.adc[c.peak] >= 8.0) and np.all(c.charge >= d.adc[c.peak])
    assert np.all(np.abs(c.pad - d.pad[c.peak]) < 1.0) and np.all(np.abs(c.time - d.time[c.peak]) < 1.0)
    assert np.all(np.diff(c.peak) > 0) and np.array_equal(c.row, d.row[c.peak].astype(np.float32))
    cell = {(int(r), int(p), int(t)) for r, p, t in zip(d.row[c.peak], d.pad[c.peak], d.time[c.peak])}
    for (r, p, t) in list(cell)[:20000]:
        assert not any((r, p + dp, t + dt) in cell for dp in (-1, 0, 1) for dt in (-1, 0, 1) if (dp, dt) != (0, 0))
    # D-E: generated clusters with no other cluster within 3 cells are found again, close to where they were put
    key = lambda r, p, t: (r.astype(np.int64) << 40) | (np.rint(t).astype(np.int64) << 12) | np.rint(p).astype(np.int64)
    gk = key(tf.row, tf.pad, tf.time)
    order = np.argsort(gk)
    gs = gk[order]
    # isolation: nearest generated neighbour in the same row farther than 3 cells in pad or time (checked on a sample)
    rng = np.random.default_rng(1)
    sample = rng.choice(tf.n, size=min(tf.n, 4000), replace=False)
    found = close = iso = 0
    ck = {}
    for i, (r, p, t) in enumerate(zip(c.row, c.pad, c.time)):
        ck.setdefault((int(r), int(np.rint(p)), int(np.rint(t))), i)
    by_row = {}
    for i in sample:
        r = int(tf.row[i])
        if r not in by_row:
            m = np.nonzero(tf.row == np.float32(r))[0]
            by_row[r] = (tf.pad[m], tf.time[m])
        pp, tt = by_row[r]
        near = (np.abs(pp - tf.pad[i]) < 3.5) & (np.abs(tt - tf.time[i]) < 3.5)
        if near.sum() != 1 or tf.charge[i] < 40:
            continue
        iso += 1
        j = ck.get((r, int(np.rint(tf.pad[i])), int(np.rint(tf.time[i]))))
        if j is None:
            continue
        found += 1
        close += abs(float(c.pad[j]) - float(tf.pad[i])) < 0.15 and abs(float(c.time[j]) - float(tf.time[i])) < 0.15
    assert iso > 300 and found >= 0.99 * iso and close >= 0.97 * found, (iso, found, close)
