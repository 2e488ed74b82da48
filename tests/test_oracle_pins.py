"""Pins of the oracle against what the paper's configuration and the mathematics fix (CPU only).

The paper prints no worked numbers for this path (PAPER.md has no tables / equations), so each pin is a
closed form, an invariant, a textbook special case or brute force on a tiny input -- SURVEY.md §8(c) table
"What pins each part" (G1, N1-N3, K1-K4, S1, E1) and BASELINE.json L5 (a)-(d).
"""
import math

import numpy as np
import pytest

import oracle
from helpers import N_ROWS, PITCH, X0, ZBIN, clusters_from_xyz, concat, n_pads, row_x
from paper_2102_08862_b200 import gen
import truth_eval

CB = 1.0 / 666.7


def _geom(n_sectors=1, tmax=487.0):
    return oracle.default_geometry(n_sectors, tmax)


# ----------------------------------------------------------------------------- G1 geometry closed forms
def test_G1_geometry_closed_forms():
    """BASELINE.json L7: x_r = 85.0 + 1.07 r, pads = floor(2 x_r tan10 / 0.5), 0.516 cm time bins over 250 cm."""
    x, npads, cr, k = oracle.tables(_geom(), oracle.default_params())
    assert npads[0] == 59 and npads[151] == 173
    assert int(npads.sum()) == 17698
    assert abs(float(x[151]) - 246.57) < 1e-4
    assert abs(250.0 / 0.516 - 484.496) < 1e-3
    np.testing.assert_array_equal(npads, n_pads(np.arange(152)))
    np.testing.assert_allclose(cr, 0.5 * (npads - 1))
    # derived constants: W1 = 0.05*1.07+0.5, A = slope*1.07 + W1, w = 1/(6 sigma^2), r = sigma^2
    assert abs(k["W1"] - 0.5535) < 1e-6 and abs(k["Ay"] - 1.6235) < 1e-6 and abs(k["Az"] - 2.1585) < 1e-6
    assert abs(k["wy"] - 1 / (6 * 0.08 ** 2)) < 1e-4 and abs(k["wz"] - 1 / (6 * 0.12 ** 2)) < 1e-4
    assert abs(k["ry"] - 0.0064) < 1e-9 and abs(k["rz"] - 0.0144) < 1e-9


# ----------------------------------------------------------------------------- K1 / K2 transport
def _state(x, y, z, s, t, k):
    return [x, y, z, s, t, k], [0.01, 0, 0.01, 0, 0, 1.0, 0.01, 0, 0.01]


@pytest.mark.parametrize("s0,k,dx", [(0.1, 2.0, 1.07), (-0.4, -4.0, 10.7), (0.6, 1.0, 50.0), (0.0, 5.0, 30.0),
                                     (0.3, 0.0, 100.0), (-0.7, 3.3, 20.0)])
def test_K1_transport_matches_exact_circle(s0, k, dx):
    """y(x) of the fp32 transport equals the circle sin(phi)(x) = s0 + kappa (x - x0) integrated in double."""
    p = oracle.default_params()
    st, cv = _state(100.0, 3.0, 0.0, s0, 0.5, k)
    ok, st1, _ = oracle.transport(p, st, cv, 100.0 + dx)
    assert ok
    kappa = float(np.float32(CB)) * k
    s1 = s0 + kappa * dx
    if kappa != 0.0:
        y_exact = 3.0 + (math.sqrt(1 - s0 * s0) - math.sqrt(1 - s1 * s1)) / kappa
        arc = (math.asin(s1) - math.asin(s0)) / kappa
    else:
        y_exact = 3.0 + dx * s0 / math.sqrt(1 - s0 * s0)
        arc = dx / math.sqrt(1 - s0 * s0)
    assert abs(float(st1[1]) - y_exact) < 1e-5 * max(1.0, abs(y_exact))
    assert abs(float(st1[3]) - s1) < 2e-7
    # K2: arc length (z advances by t * dS with t = 0.5): series vs asin form, < 1e-6 relative when kappa*chord <= 0.3
    chord = math.hypot(dx, y_exact - 3.0)
    assert abs(kappa) * chord <= 0.3
    assert abs(float(st1[2]) / 0.5 - arc) < 2e-6 * abs(arc)


def test_K2_arc_series_coefficients():
    """arc/chord = (2/a) asin(a/2) = 1 + a^2/24 + 3a^4/640 + 5a^6/7168 + ...: relative error < 1e-6 for a <= 0.3."""
    for a in np.linspace(1e-3, 0.3, 50):
        q = a * a
        series = 1 + q * (0.041666668 + q * (0.0046875 + q * 0.00069754466))
        assert abs(series - (2 / a) * math.asin(a / 2)) < 1e-6


def test_K1_transport_round_trip_and_composition():
    p = oracle.default_params()
    st, cv = _state(90.0, -2.0, 1.0, 0.25, -0.8, 3.0)
    ok1, a, ca = oracle.transport(p, st, cv, 120.0)
    ok2, b, _ = oracle.transport(p, a, ca, 90.0)
    assert ok1 and ok2
    np.testing.assert_allclose(b, np.array(st, np.float32), atol=3e-5, rtol=3e-6)
    ok3, c, _ = oracle.transport(p, a, ca, 160.0)
    ok4, d, _ = oracle.transport(p, st, cv, 160.0)
    assert ok3 and ok4
    np.testing.assert_allclose(c, d, atol=5e-5, rtol=5e-6)


def test_K1_transport_fails_beyond_sin_phi_max_and_keeps_state():
    p = oracle.default_params()
    st, cv = _state(90.0, 0.0, 0.0, 0.9, 0.0, 10.0)     # s grows by cB*k*dx = 0.015/cm
    ok, st1, cv1 = oracle.transport(p, st, cv, 100.0)
    assert not ok
    np.testing.assert_array_equal(st1, np.array(st, np.float32))
    np.testing.assert_array_equal(cv1, np.array(cv, np.float32))


def test_K1_sin_phi_exactly_on_the_limit_fails_at_either_end():
    """A12: the step needs |sin phi| < sin_phi_max at BOTH ends, strictly (all values below are exact in fp32)."""
    p = oracle.default_params()
    p.sin_phi_max = 0.75
    p.inv_R_per_qpt = 0.5
    cv = [1, 0, 1, 0, 0, 1, 1, 0, 1]
    ok, st, _ = oracle.transport(p, [100.0, 0.0, 0.0, 0.75, 0.0, 0.0], cv, 101.0)             # starts on the limit
    assert not ok and st[0] == 100.0
    ok, st, _ = oracle.transport(p, [100.0, 0.0, 0.0, 0.5, 0.0, 0.5], cv, 101.0)              # ends on it: 0.5 + 0.5 * 0.5 * 1
    assert not ok and st[0] == 100.0
    ok, st, _ = oracle.transport(p, [100.0, 0.0, 0.0, 0.5, 0.0, 0.5], cv, 100.96875)          # ends just inside
    assert ok and st[3] == np.float32(0.5 + 0.25 * 0.96875)
    ok, st, _ = oracle.transport(p, [100.0, 0.0, 0.0, -0.75, 0.0, 0.0], cv, 101.0)
    assert not ok


def test_K1_transport_never_leaves_the_domain_of_the_circle():
    """Reading A12 on both ends: whatever an update did to sin phi (even |s| >= 1, where sqrt(1 - s^2) does not exist),
    a transport either FAILs and keeps the state or returns finite numbers."""
    rng = np.random.default_rng(17)
    p = oracle.default_params()
    p.sin_phi_max = 0.99
    n_fail = n_ok = 0
    for _ in range(3000):
        st = [rng.uniform(85, 245), rng.uniform(-40, 40), rng.uniform(-100, 100), rng.uniform(-1.3, 1.3), rng.uniform(-1.5, 1.5), rng.uniform(-30, 30)]
        ok, a, c = oracle.transport(p, st, [1, 0, 0.1, 0, 0, 100, 1, 0, 0.1], st[0] + rng.uniform(-12, 12))
        assert np.all(np.isfinite(a)) and np.all(np.isfinite(c))
        if abs(st[3]) >= 0.99:
            assert not ok
        if not ok:
            np.testing.assert_array_equal(a, np.array(st, np.float32))
        n_fail += (not ok); n_ok += ok
    assert n_fail > 300 and n_ok > 300


def test_K1_covariance_transport_is_F_C_Ft():
    """The staged covariance lines equal F C F^T with the Jacobian taken by finite differences in double."""
    p = oracle.default_params()
    rng = np.random.default_rng(5)
    A = rng.normal(size=(3, 3)); CA = A @ A.T * 1e-3
    B = rng.normal(size=(2, 2)); CBk = B @ B.T * 1e-3
    cov = [CA[0, 0], CA[0, 1], CA[1, 1], CA[0, 2], CA[1, 2], CA[2, 2], CBk[0, 0], CBk[0, 1], CBk[1, 1]]
    x0, y0, s0, k0, dx = 100.0, 1.0, 0.3, 2.5, 12.0
    ok, _, cv1 = oracle.transport(p, [x0, y0, 0.0, s0, 0.4, k0], cov, x0 + dx)
    assert ok

    def prop(v):   # exact circle, double
        y, s, k = v
        kap = CB * k
        s1 = s + kap * dx
        return np.array([y + dx * (s + s1) / (math.sqrt(1 - s * s) + math.sqrt(1 - s1 * s1)), s1, k])

    F = np.zeros((3, 3)); v0 = np.array([y0, s0, k0])
    for j in range(3):
        e = np.zeros(3); e[j] = 1e-6
        F[:, j] = (prop(v0 + e) - prop(v0 - e)) / 2e-6
    CA1 = F @ CA @ F.T
    got = np.array([[cv1[0], cv1[1], cv1[3]], [cv1[1], cv1[2], cv1[4]], [cv1[3], cv1[4], cv1[5]]], np.float64)
    np.testing.assert_allclose(got, CA1, rtol=2e-4, atol=1e-8)
    s1 = s0 + CB * k0 * dx
    dS = (math.asin(s1) - math.asin(s0)) / (CB * k0)
    Fz = np.array([[1, dS], [0, 1]])
    CB1 = Fz @ CBk @ Fz.T
    np.testing.assert_allclose([cv1[6], cv1[7], cv1[8]], [CB1[0, 0], CB1[0, 1], CB1[1, 1]], rtol=2e-4, atol=1e-8)


# ----------------------------------------------------------------------------- K3 filter == least squares
def test_K3_filter_equals_weighted_least_squares_line():
    """With the curvature frozen (k = 0, c3 = c4 = c5 = 0) the filter is the textbook weighted least-squares
    straight-line fit with a Gaussian prior (normal equations (A^T A / r + P0^-1)^-1 A^T z / r): exactly linear
    in the (z, t) block.  A prior of 100 keeps fp32 cancellation in c - k*c below the tolerance."""
    p = oracle.default_params()
    rng = np.random.default_rng(11)
    xs = X0 + PITCH * np.arange(40)
    zt, tt = 2.0, 0.7
    zm = zt + tt * (xs - xs[0]) + rng.normal(0, 0.12, xs.size)
    ym = 0.5 + 0.01 * (xs - xs[0]) + rng.normal(0, 0.01, xs.size)
    P0 = 100.0
    st = np.array([xs[0], 0.0, 0.0, 0.0, 0.0, 0.0], np.float32)
    cv = np.array([P0, 0, P0, 0, 0, 0, P0, 0, P0], np.float32)
    ry, rz = 0.01 ** 2, 0.12 ** 2
    for i, x in enumerate(xs):
        if i:
            ok, st, cv = oracle.transport(p, st, cv, float(x))
            assert ok
        st, cv = oracle.update(st, cv, float(ym[i]), float(zm[i]), ry, rz)

    def bayes_line(u, meas, r):
        A = np.stack([np.ones_like(u), u], 1)
        cov = np.linalg.inv(A.T @ A / r + np.eye(2) / P0)
        return cov @ (A.T @ meas / r), cov

    # z block: the path length per step is dx*sqrt(1+T^2) with T = tan(phi) ~ 0.01
    T = 0.01
    sl = (xs - xs[0]) * math.sqrt(1 + T * T)
    (z_ls, t_ls), cov = bayes_line(sl, zm, rz)
    a = np.array([1.0, sl[-1]])
    assert abs(float(st[2]) - (z_ls + t_ls * sl[-1])) < 1e-4 and abs(float(st[4]) - t_ls) < 1e-5
    assert abs(float(cv[6]) - a @ cov @ a) < 2e-3 * (a @ cov @ a)
    assert abs(float(cv[8]) - cov[1, 1]) < 2e-3 * cov[1, 1]
    # y block: a line in tan(phi); the filter's parameter is s = sin(phi) (linearisation error ~ T^2)
    (y_ls, sl_ls), _ = bayes_line(xs - xs[0], ym, ry)
    assert abs(float(st[1]) - (y_ls + sl_ls * (xs[-1] - xs[0]))) < 1e-4
    assert abs(float(st[3]) - sl_ls / math.sqrt(1 + sl_ls ** 2)) < 1e-5


# ----------------------------------------------------------------------------- N2 straight tracks
def _straight_tracks(n_tracks=6, seed=3):
    rng = np.random.default_rng(seed)
    rows = np.arange(N_ROWS)
    x = row_x(rows)
    parts = []
    for i in range(n_tracks):      # radial-ish lines that stay inside the +-10 degree wedge and the drift length
        y = (-0.12 + 0.048 * i) * x + rng.uniform(-0.01, 0.01) * (x - X0)
        z = 125.0 + rng.uniform(-0.7, 0.7) * (x - X0)
        parts.append(clusters_from_xyz(rows, y, z))
    return concat(parts), n_tracks


def test_N2_noise_free_straight_tracks_link_to_true_neighbours():
    (row, pad, time), nt = _straight_tracks()
    r = oracle.track(_geom(), oracle.default_params(), row, pad, time)
    idx = np.arange(row.size).reshape(nt, N_ROWS)
    for t in range(nt):
        # uncleaned: every interior hit links to the hits of its own track in rows r+1 and r-1
        np.testing.assert_array_equal(r.up_raw[idx[t, 1:-1]], idx[t, 2:])
        np.testing.assert_array_equal(r.down_raw[idx[t, 1:-1]], idx[t, :-2])
        # edge rows are linkless, so after cleaning the chain is rows 1..150 and row 1 is the only start hit
        assert r.link_up[idx[t, 150]] == -1 and r.link_down[idx[t, 1]] == -1
        np.testing.assert_array_equal(r.link_up[idx[t, 1:150]], idx[t, 2:151])
        assert r.is_start_hit[idx[t]].sum() == 1 and r.is_start_hit[idx[t, 1]] == 1
    # BASELINE.json L5 (a): reconstructed exactly -- one track per line with all 152 hits
    assert len(r.tr_seed) == nt
    for i in range(nt):
        t = int(np.where(idx[:, 1] == r.tr_seed[i])[0][0])
        np.testing.assert_array_equal(r.track_hits(i), idx[t])
        assert abs(float(r.tr_par[i, 5])) < 2e-2          # q/pT ~ 0 for a straight line


# ----------------------------------------------------------------------------- N1 brute force
def _small_frame(seed, n_tracks=40, **kw):
    c = gen.preset(0, seed)
    c.fixed_tracks = n_tracks
    for k, v in kw.items():
        setattr(c, k, v)
    return gen.generate(c)


def _numpy_all_pairs_links(row, pad, time, consts, npads_tab, chi2_cut):
    """C2 by brute force over ALL hits of rows r+1 / r-1 in fp32 numpy (tiny inputs only)."""
    f = np.float32
    sr = row.astype(np.int64)
    r = sr % N_ROWS
    y = ((pad - (0.5 * (npads_tab[r] - 1)).astype(f)) * f(0.5)).astype(f)
    n = row.size
    up = np.full(n, -1, np.int32); dn = np.full(n, -1, np.int32)
    Z = f(ZBIN)
    for h in range(n):
        if r[h] < 1 or r[h] > N_ROWS - 2:
            continue
        best = None
        for u in np.where(sr == sr[h] + 1)[0]:
            if not (abs(f(y[u] - y[h])) < consts["Ay"] and abs(f(f(time[u] - time[h]) * Z)) < consts["Az"]):
                continue
            for d in np.where(sr == sr[h] - 1)[0]:
                if not (abs(f(y[d] - y[h])) < consts["Ay"] and abs(f(f(time[d] - time[h]) * Z)) < consts["Az"]):
                    continue
                ey = f(f(y[u] - y[h]) - f(y[h] - y[d]))
                ez = f(f(f(time[u] - time[h]) * Z) - f(f(time[h] - time[d]) * Z))
                if not (abs(ey) < consts["W1"] and abs(ez) < consts["W1"]):
                    continue
                chi2 = f(f(f(ey * ey) * consts["wy"]) + f(f(ez * ez) * consts["wz"]))
                if not chi2 < chi2_cut:
                    continue
                key = (chi2, u, d)
                if best is None or key < best:
                    best = key
        if best is not None:
            up[h], dn[h] = best[1], best[2]
    return up, dn


def test_N1_brute_force_equals_window_search():
    """BASELINE.json L5 (b): brute-force all-pairs neighbour search agrees with the windowed search."""
    tf = _small_frame(7, n_tracks=12)
    assert tf.n <= 2000
    g, p = _geom(1, tf.max_time_bin), oracle.default_params()
    fast = oracle.track(g, p, tf.row, tf.pad, tf.time)
    p.brute_force = 1
    brute = oracle.track(g, p, tf.row, tf.pad, tf.time)
    for name in ("up_raw", "down_raw", "link_up", "link_down", "is_start_hit", "tl_row_hit", "tr_hit_index", "tr_par"):
        np.testing.assert_array_equal(getattr(fast, name), getattr(brute, name), err_msg=name)
    # and against an independent all-pairs evaluation in numpy fp32 (tie-breaks on original index)
    _, npads_tab, _, consts = oracle.tables(g, p)
    up, dn = _numpy_all_pairs_links(tf.row, tf.pad, tf.time, consts, npads_tab, np.float32(9.0))
    np.testing.assert_array_equal(fast.up_raw, up)
    np.testing.assert_array_equal(fast.down_raw, dn)
    assert (up >= 0).sum() > 200


def test_N1_ties_break_on_lowest_original_index():
    """Two identical candidates in the upper row: the link goes to the lower original index, wherever it sits."""
    rows = np.array([10, 11, 12, 12])
    base = clusters_from_xyz(rows, [0.0, 0.1, 0.2, 0.2], [50.0, 50.5, 51.0, 51.0])
    for perm in ([0, 1, 2, 3], [3, 2, 1, 0], [2, 0, 3, 1]):
        row, pad, time = (a[perm] for a in base)
        r = oracle.track(_geom(), oracle.default_params(), row, pad, time)
        h = perm.index(1)
        dup = sorted([perm.index(2), perm.index(3)])
        assert r.up_raw[h] == dup[0] and r.down_raw[h] == perm.index(0)


# ----------------------------------------------------------------------------- N3 / invariants
@pytest.mark.parametrize("seed", [1, 2])
def test_N3_invariants(seed):
    """BASELINE.json L5 (c): links reciprocal after cleaning, each hit in at most one track, counts conserved."""
    tf = _small_frame(seed, n_tracks=150)
    r = oracle.track(_geom(1, tf.max_time_bin), oracle.default_params(), tf.row, tf.pad, tf.time)
    h = np.where(r.link_up >= 0)[0]
    np.testing.assert_array_equal(r.link_down[r.link_up[h]], h)
    h = np.where(r.link_down >= 0)[0]
    np.testing.assert_array_equal(r.link_up[r.link_down[h]], h)
    # links join adjacent rows of the same sector
    sr = tf.row.astype(np.int64)
    h = np.where(r.link_up >= 0)[0]
    np.testing.assert_array_equal(sr[r.link_up[h]], sr[h] + 1)
    # start hits: no down link, chain of >= 3
    s = np.where(r.is_start_hit)[0]
    assert (r.link_down[s] < 0).all()
    assert (r.link_up[s] >= 0).all() and (r.link_up[r.link_up[s]] >= 0).all()
    np.testing.assert_array_equal(np.sort(s), np.sort(r.tl_seed))
    # each hit in at most one final track; hit counts conserved
    assert np.unique(r.tr_hit_index).size == r.tr_hit_index.size
    assert int(r.tr_n_hits.sum()) == r.tr_hit_index.size
    assert (r.tr_n_hits >= 30).all()
    for i in range(len(r.tr_seed)):
        hits = r.track_hits(i)
        rows = sr[hits] % N_ROWS
        assert (np.diff(rows) > 0).all()                       # ascending row, one hit per row
        assert rows[0] == r.tr_first_row[i] and rows[-1] == r.tr_last_row[i]
        t = int(np.where(r.tl_seed == r.tr_seed[i])[0][0])
        assert set(hits.tolist()) <= set(r.tl_row_hit[t][r.tl_row_hit[t] >= 0].tolist())
    # tracklet bookkeeping
    np.testing.assert_array_equal((r.tl_row_hit >= 0).sum(1), r.tl_n_hits)


# ----------------------------------------------------------------------------- S1 selector
def test_S1_selector_equals_sorted_first_come_first_served():
    tf = _small_frame(4, n_tracks=200)
    p = oracle.default_params()
    r = oracle.track(_geom(1, tf.max_time_bin), p, tf.row, tf.pad, tf.time)
    cand = [i for i in range(len(r.tl_seed)) if r.tl_n_hits[i] >= p.min_hits]
    cand.sort(key=lambda i: (-int(r.tl_n_hits[i]), int(r.tl_seed[i])))      # key (nHits, -id) descending
    owner = {}
    for i in cand:
        for hidx in r.tl_row_hit[i][r.tl_row_hit[i] >= 0]:
            owner.setdefault(int(hidx), i)
    expect = {}
    for i in cand:
        own = [int(hidx) for hidx in r.tl_row_hit[i] if hidx >= 0 and owner[int(hidx)] == i]
        if len(own) >= p.min_hits:
            expect[int(r.tl_seed[i])] = own
    assert len(expect) > 20
    assert sorted(expect) == sorted(r.tr_seed.tolist())
    for i in range(len(r.tr_seed)):
        assert expect[int(r.tr_seed[i])] == r.track_hits(i).tolist()
        t = int(np.where(r.tl_seed == r.tr_seed[i])[0][0])
        np.testing.assert_array_equal(r.tr_par[i], r.tl_par[t])             # parameters unchanged, no refit


# ----------------------------------------------------------------------------- K4 noise-free helices
def test_K4_noise_free_helices_reconstructed_exactly():
    """BASELINE.json L5 (a): noise-free helix tracks are reconstructed exactly."""
    tf = _small_frame(9, n_tracks=12, sigma_y_cm=0.0, sigma_z_cm=0.0, dropout=0.0, noise_frac=0.0, pt_min=0.4)
    p = oracle.default_params()
    r = oracle.track(_geom(1, tf.max_time_bin), p, tf.row, tf.pad, tf.time)
    seg = truth_eval.segment_ids(tf)
    useg, cnt = np.unique(seg, return_counts=True)
    long_segs = useg[cnt >= 40]
    assert len(long_segs) >= 8
    seg_of_track = {}
    for i in range(len(r.tr_seed)):
        s = np.unique(seg[r.track_hits(i)])
        assert s.size == 1                                                   # pure
        assert int(s[0]) not in seg_of_track                                 # no clones
        seg_of_track[int(s[0])] = i
    x_r = row_x(np.arange(N_ROWS))
    for s in long_segs:
        i = seg_of_track[int(s)]
        hits = np.sort(np.where(seg == s)[0])
        np.testing.assert_array_equal(np.sort(r.track_hits(i)), hits)        # exactly all its hits
        tr = tf.tracks[int(s) // (64 * 16)]
        qpt_true = tr["charge_sense"] / tr["pt"]
        assert abs(float(r.tr_par[i, 5]) / qpt_true - 1.0) < 1e-3
        # state at the innermost hit reproduces that hit and the true local direction
        first = r.track_hits(i)[0]
        row0 = int(tf.row[first]) % N_ROWS
        y0 = (float(tf.pad[first]) - 0.5 * (n_pads(row0) - 1)) * 0.5
        assert abs(float(r.tr_par[i, 1]) - y0) < 1e-4
        sin_true = math.sin(tr["phi0"]) + tr["charge_sense"] * x_r[row0] / (666.7 * tr["pt"])
        assert abs(float(r.tr_par[i, 3]) - sin_true) < 1e-4
        z_rel_true = (float(tf.time[first]) - float(r.tr_par[i, 6])) * ZBIN
        assert abs(float(r.tr_par[i, 2]) - z_rel_true) < 1e-4


# ----------------------------------------------------------------------------- E1 efficiency
@pytest.mark.parametrize("cid,seed", [(0, 1), (0, 2), (1, 1)])
def test_E1_efficiency_at_least_95_percent(cid, seed):
    """BASELINE.json L5 (d): efficiency >= 95 % against generator truth for pT > 0.2 GeV."""
    cfg = gen.preset(cid, seed)
    tf = gen.generate(cfg)
    r = oracle.track(oracle.default_geometry(cfg.n_sectors, tf.max_time_bin),
                     oracle.default_params(cfg.sigma_y_cm, cfg.sigma_z_cm), tf.row, tf.pad, tf.time)
    e = truth_eval.evaluate(tf, r.tr_hit_offset, r.tr_n_hits, r.tr_hit_index)
    assert e["n_findable"] >= 50
    assert e["efficiency"] >= 0.95, e
    assert e["fake_rate"] <= 0.02 and e["clone_rate"] <= 0.02, e


# ----------------------------------------------------------------------------- P1..P4: hand-built pins of the cuts
# Each of these exists because a plausible one-token mistake in the oracle survived every pin above (round-1 review):
# the follower's stop rule, the growth of its window over missed rows, the two bounds of the finder's search area and
# the seed's dz/ds.  All inputs are noise-free straight lines, so the expected outcome follows from BASELINE.json L7's
# cuts ("0.05*dx + 0.5 cm" windows, "miss limit of 10 consecutive missed rows") by hand.
def _line(rows, slope_y=0.02, slope_z=0.3, y_at=0.0, z_at=150.0, dy=0.0, dz=0.0):
    """Clusters of the straight line y = y_at + slope_y (x - x0), z = z_at + slope_z (x - x0) at the given rows,
    every one displaced by (dy, dz)."""
    rows = np.asarray(rows)
    x = row_x(rows)
    return clusters_from_xyz(rows, y_at + slope_y * (x - X0) + dy, z_at + slope_z * (x - X0) + dz)


def _track_one(parts, **params):
    row, pad, time = concat(parts)
    p = oracle.default_params()
    for k, v in params.items():
        setattr(p, k, v)
    return oracle.track(_geom(), p, row, pad, time), row


@pytest.mark.parametrize("gap,bridged", [(9, True), (10, False)])
def test_P1_miss_limit_upward_is_the_tenth_consecutive_missed_row(gap, bridged):
    """BASELINE.json L7 "a miss limit of 10 consecutive missed rows ends track following" (reading A11): a gap of 9 rows
    is crossed, the 10th consecutive missed row ends the direction.  Above the gap only two hits (no chain of three, so
    nothing but the follower of the lower piece can pick them up)."""
    lower = np.arange(20, 61)
    upper = np.array([61 + gap, 62 + gap])
    r, row = _track_one([_line(lower), _line(upper)])
    assert len(r.tl_seed) == 1 and len(r.tr_seed) == 1
    got = np.sort((row[r.track_hits(0)]).astype(int))
    want = np.concatenate([lower, upper]) if bridged else lower
    np.testing.assert_array_equal(got, want)


@pytest.mark.parametrize("gap,bridged", [(9, True), (10, False)])
def test_P1_miss_limit_downward_is_the_tenth_consecutive_missed_row(gap, bridged):
    """The same rule in the down pass below the seed row."""
    upper = np.arange(80, 121)
    lower = np.array([78 - gap, 79 - gap])
    r, row = _track_one([_line(upper), _line(lower)])
    assert len(r.tl_seed) == 1 and len(r.tr_seed) == 1
    got = np.sort((row[r.track_hits(0)]).astype(int))
    want = np.concatenate([lower, upper]) if bridged else upper
    np.testing.assert_array_equal(got, want)


def test_P1_a_hit_resets_the_miss_count_and_holes_in_the_refit_are_not_misses():
    """Three gaps of 9 rows in a row: the count is of CONSECUTIVE misses (a hit resets it), and in the down pass the 27
    holes inside the collected range do not count at all (reading A11, second half)."""
    rows = np.concatenate([np.arange(10, 51), [60], [70], [80, 81]])
    r, row = _track_one([_line(rows)])
    assert len(r.tr_seed) == 1
    np.testing.assert_array_equal(np.sort(row[r.track_hits(0)].astype(int)), rows)


@pytest.mark.parametrize("axis", ["y", "z"])
@pytest.mark.parametrize("k_missed,disp,attached", [(5, 0.70, True), (5, 0.90, False), (0, 0.50, True), (0, 0.60, False),
                                                    (8, 0.90, True), (8, 1.06, False)])
def test_P2_follower_window_grows_with_the_distance_since_the_last_hit(axis, k_missed, disp, attached):
    """BASELINE.json L7 "0.05*dx + 0.5 cm" with dx = distance since the last attached hit (reading A1): after k missed
    rows the window is W = 0.05 * 1.07 (k + 1) + 0.5 (0.5535, 0.821, 0.9815 for k = 0, 5, 8).  A single hit displaced
    by `disp` from the line is attached iff disp < W, in y and in z alike."""
    lower = np.arange(20, 61)
    far = np.array([61 + k_missed])
    w = 0.05 * 1.07 * (k_missed + 1) + 0.5
    assert (disp < w) == attached and abs(disp - w) > 0.04          # the case is not marginal
    kw = {"dy": disp} if axis == "y" else {"dz": disp}
    r, row = _track_one([_line(lower), _line(far, **kw)])
    assert len(r.tr_seed) == 1
    got = np.sort(row[r.track_hits(0)].astype(int))
    np.testing.assert_array_equal(got, np.concatenate([lower, far]) if attached else lower)


def test_P3_search_area_bounds_y_and_z_separately():
    """The finder's search area is |dy| < A_y = slope_y_max*1.07 + W1 (1.6235) and |dz| < A_z = slope_z_max*1.07 + W1
    (2.1585) (reading A1).  A perfect straight line stepping 1.9 cm per row links when the step is
    in z and does not when it is in y; 1.5 cm links in both; 2.3 cm in neither."""
    rows = np.arange(40, 47)
    for step, in_y, in_z in ((1.9, False, True), (1.5, True, True), (2.3, False, False)):
        for axis, expect in (("y", in_y), ("z", in_z)):
            kw = dict(slope_y=step / PITCH, slope_z=0.0, y_at=-5.0 - 40 * step) if axis == "y" else dict(slope_y=0.0, slope_z=step / PITCH)
            row, pad, time = _line(rows, **kw)
            r = oracle.track(_geom(1, 1200.0), oracle.default_params(), row, pad, time)
            linked = r.up_raw[1:-1] >= 0
            assert linked.all() == expect and linked.any() == expect, (step, axis)
            if expect:
                np.testing.assert_array_equal(r.up_raw[1:-1], np.arange(2, rows.size))
                np.testing.assert_array_equal(r.down_raw[1:-1], np.arange(0, rows.size - 2))


def test_N1_brute_force_on_steep_tracks():
    """N1 again on hand-made steep lines (|dy/dx| up to 1.4, |dz/dx| up to 1.9: candidates between the two bounds of
    the search area exist) plus uniform noise, against the independent numpy all-pairs evaluation."""
    rng = np.random.default_rng(21)
    rows = np.arange(30, 52)
    parts = []
    for sy, sz in ((1.4, 0.2), (-1.3, 1.9), (0.9, -1.7), (1.45, 1.45), (0.1, 1.95), (-1.0, -0.4)):
        parts.append(_line(rows, slope_y=sy, slope_z=sz, y_at=-sy * (row_x(41) - X0), z_at=120.0))
    nr = rng.integers(30, 52, 250)
    parts.append(((nr).astype(np.float32), rng.uniform(5, 60, 250).astype(np.float32), rng.uniform(150, 330, 250).astype(np.float32)))
    row, pad, time = concat(parts)
    g, p = _geom(1, 600.0), oracle.default_params()
    fast = oracle.track(g, p, row, pad, time)
    _, npads_tab, _, consts = oracle.tables(g, p)
    up, dn = _numpy_all_pairs_links(row, pad, time, consts, npads_tab, np.float32(9.0))
    np.testing.assert_array_equal(fast.up_raw, up)
    np.testing.assert_array_equal(fast.down_raw, dn)
    assert (up >= 0).sum() >= 6 * 18
    # the steep-in-y lines link (1.4 * 1.07 + noise-free < A_y), so candidates beyond A_y but inside A_z were rejected
    x = row_x(rows)
    assert 1.45 * PITCH < 1.6235 < 1.9 * PITCH < 2.1585


def test_P4_seed_state_is_direction_cosines_of_the_first_two_hits():
    """C5 step 1 (reading A7): s = dy/L, t = dz/L with L = sqrt(dx^2 + dy^2) -- BOTH over the path length in the bending
    plane.  With sin_phi_max lowered below the seed's sin phi the very first transport FAILs, so the tracklet's output
    IS the init state: x = x_r0, y = y(h0), z = 0, s = 0.6, t = 0.8, k = 0 for a line with dy/dx = 0.75, dz/dx = 1."""
    rows = np.arange(10, 15)
    row, pad, time = _line(rows, slope_y=0.75, slope_z=1.0, y_at=-12.0, z_at=100.0)
    p = oracle.default_params()
    p.sin_phi_max = 0.5
    r = oracle.track(_geom(), p, row, pad, time)
    assert len(r.tl_seed) == 1 and r.tl_seed[0] == 1 and r.tl_n_hits[0] == 1      # start hit = row 11 (row 10 is linkless)
    par = r.tl_par[0].astype(np.float64)
    y0 = (float(pad[1]) - 0.5 * (n_pads(11) - 1)) * 0.5
    assert abs(par[0] - row_x(11)) < 1e-4 and abs(par[1] - y0) < 1e-5 and par[2] == 0.0 and par[5] == 0.0
    assert abs(par[3] - 0.6) < 2e-4           # pads are fp32: the line is reproduced to ~1e-5 cm
    assert abs(par[4] - 0.8) < 2e-4           # dz/dx (= 1.0) here would be the mistake
    assert par[6] == time[1]


def test_N1_tie_between_equal_lower_candidates_goes_to_the_lower_original_index():
    """C2's second tie level: the same upper hit, two identical candidates in the LOWER row."""
    rows = np.array([10, 10, 11, 12])
    base = clusters_from_xyz(rows, [0.0, 0.0, 0.1, 0.2], [50.0, 50.0, 50.5, 51.0])
    for perm in ([0, 1, 2, 3], [3, 2, 1, 0], [1, 3, 0, 2]):
        row, pad, time = (a[perm] for a in base)
        r = oracle.track(_geom(), oracle.default_params(), row, pad, time)
        h = perm.index(2)
        dup = sorted([perm.index(0), perm.index(1)])
        assert r.up_raw[h] == perm.index(3) and r.down_raw[h] == dup[0]


def test_P5_search_tie_goes_to_the_lower_original_index():
    """C5 search: two identical hits in a followed row (not part of the seed chain): the tracklet takes the lower original
    index, wherever the two sit in the input."""
    lower, upper = np.arange(20, 46), np.arange(48, 61)
    parts = [_line(lower), _line(upper), _line(np.array([50]))]               # row 50 twice
    row, pad, time = concat(parts)
    n = row.size
    for perm in (np.arange(n), np.arange(n)[::-1], np.random.default_rng(4).permutation(n)):
        r = oracle.track(_geom(), oracle.default_params(), row[perm], pad[perm], time[perm])
        dup = np.nonzero(row[perm] == 50.0)[0]
        assert dup.size == 2
        seed_rows = row[perm][r.tl_seed].astype(int)
        t = int(np.nonzero(seed_rows == 21)[0][0])                                 # the tracklet seeded in the lower part: it SEARCHES row 50
        assert r.tl_row_hit[t, 50] == dup.min(), (r.tl_row_hit[t, 50], dup)
        assert r.tl_row_hit[t, 46] == -1 and r.tl_row_hit[t, 48] >= 0


def test_P6_holes_inside_the_collected_range_are_not_searched_again_on_the_way_down():
    """Reading A13: the down pass refits through the collected hits and searches only BELOW the seed row.  A hit displaced
    by 0.58 cm sits in a hole of the up pass (window 0.5535 cm one row after a hit); on the way down the last update is two
    rows away (window 0.607 cm) -- a search there would attach it."""
    rows = np.concatenate([np.arange(20, 25), np.arange(27, 61)])               # rows 25, 26 empty on the line
    r, row = _track_one([_line(rows), _line(np.array([25]), dy=0.58)])
    t = int(np.nonzero(row[r.tl_seed].astype(int) == 21)[0][0])      # the tracklet seeded BELOW the hole: rows 25, 26 are inside its collected range
    assert r.tl_row_hit[t, 25] == -1 and r.tl_row_hit[t, 26] == -1 and r.tl_n_hits[t] == rows.size
    # (the tracklet seeded above the hole, at row 28, searches rows 27 .. 0 on its way down and does attach it: window 0.607 cm)
    t_up = int(np.nonzero(row[r.tl_seed].astype(int) == 28)[0][0])
    assert r.tl_row_hit[t_up, 25] >= 0
    # control: the same hit displaced by 0.50 cm IS attached (on the way up, window 0.5535)
    r2, _ = _track_one([_line(rows), _line(np.array([25]), dy=0.50)])
    row2 = concat([_line(rows), _line(np.array([25]), dy=0.50)])[0]
    t2 = int(np.nonzero(row2[r2.tl_seed].astype(int) == 21)[0][0])
    assert r2.tl_row_hit[t2, 25] >= 0


def test_G3_validity_bounds_of_a_cluster_are_half_open_in_pad_and_closed_in_time():
    """C1: pad in [-0.5, n_pads - 0.5) (pad p covers [p - 0.5, p + 0.5)), time in [0, max_time_bin].  A cluster exactly on a
    bound is counted or ignored accordingly (the ignored ones are reported in stats)."""
    tmax = 600.0
    line = _line(np.arange(30, 70))
    def n_invalid(pad_value, time_value, row_value=40.0):
        row = np.concatenate([line[0], [row_value]]).astype(np.float32)
        pad = np.concatenate([line[1], [pad_value]]).astype(np.float32)
        time = np.concatenate([line[2], [time_value]]).astype(np.float32)
        r = oracle.track(_geom(1, tmax), oracle.default_params(), row, pad, time)
        assert len(r.tr_seed) == 1 and r.tr_n_hits[0] == 40             # the line itself is untouched
        return int(r.stats["invalid_clusters"])
    np40 = float(n_pads(40))
    assert n_invalid(np40 - 0.5, 100.0) == 1                # the upper pad bound is excluded ...
    assert n_invalid(np.float32(np40 - 0.5) - np.float32(1e-3), 100.0) == 0
    assert n_invalid(-0.5, 100.0) == 0                      # ... the lower one included
    assert n_invalid(np.float32(-0.5) - np.float32(1e-3), 100.0) == 1
    assert n_invalid(10.0, tmax) == 0                       # time == max_time_bin is inside
    assert n_invalid(10.0, np.nextafter(np.float32(tmax), np.float32(1e9))) == 1
    assert n_invalid(10.0, 0.0) == 0 and n_invalid(10.0, -1e-3) == 1
    assert n_invalid(10.0, 100.0, row_value=152.0) == 1     # beyond the single sector
    assert n_invalid(10.0, 100.0, row_value=40.5) == 1      # not an integer row


def test_N4_edge_rows_have_no_links_even_next_to_another_sector():
    """Reading A5: rows 0 and n_rows - 1 are linkless; a link never crosses into the neighbouring sector (whose row 0 follows
    row 151 in the sector-row numbering)."""
    a = _line(np.arange(140, 152))                          # sector 0, up to its last row
    b = _line(np.arange(0, 12), y_at=float(0.02 * 1.07 * 152), z_at=150.0 + 0.3 * 1.07 * 152)   # sector 1: the SAME line continued, as rows 0..11
    b = (b[0] + np.float32(152.0), b[1], b[2])
    row, pad, time = concat([a, b])
    r = oracle.track(_geom(2, 800.0), oracle.default_params(), row, pad, time)
    i151 = int(np.nonzero(row == 151.0)[0][0]); i152 = int(np.nonzero(row == 152.0)[0][0])
    assert r.up_raw[i151] == -1 and r.down_raw[i151] == -1 and r.up_raw[i152] == -1 and r.down_raw[i152] == -1
    i150 = int(np.nonzero(row == 150.0)[0][0])
    assert r.up_raw[i150] == i151 and r.down_raw[i150] >= 0   # row 150 does link up to the edge row


# ---- pins from the line-by-line mutation sweep of orc_track ------------------------------------------------

def test_P7_search_distance_adds_the_z_term():
    """C5 search: nearest in dy^2 + dz^2.  Row 50 holds A (dy 0.30, dz 0) and B (dy 0.10, dz 0.35): dd = 0.090 against 0.1325, A
    is attached; with the z term dropped or subtracted B would be.  (Neither links in the finder: |ez| or |ey| beyond W1 on one
    side, so row 50 is reached by the follower's search -- from below and, by the tracklet seeded above, from above.)"""
    rows = np.concatenate([np.arange(20, 50), np.arange(51, 61)])
    row, pad, time = concat([_line(rows), _line(np.array([50]), dy=0.30), _line(np.array([50]), dy=0.10, dz=0.35)])
    ia, ib = rows.size, rows.size + 1
    r = oracle.track(_geom(), oracle.default_params(), row, pad, time)
    assert r.link_up[int(np.nonzero(row == 49.0)[0][0])] == -1                  # no cleaned link into row 50
    seed_rows = row[r.tl_seed].astype(int)
    for seed_row in (21, 51):
        t = int(np.nonzero(seed_rows == seed_row)[0][0])
        assert r.tl_row_hit[t, 50] == ia, (seed_row, r.tl_row_hit[t, 50], ia, ib)
    # control: B moved to dz = 0.25 is the nearer one (0.0725)
    row, pad, time = concat([_line(rows), _line(np.array([50]), dy=0.30), _line(np.array([50]), dy=0.10, dz=0.25)])
    r = oracle.track(_geom(), oracle.default_params(), row, pad, time)
    t = int(np.nonzero(row[r.tl_seed].astype(int) == 21)[0][0])
    assert r.tl_row_hit[t, 50] == ib


def test_P8_finder_chi2_adds_the_z_term():
    """C2: chi2 = ey^2 w_y + ez^2 w_z.  Above the hit of row 30 sit u1 (ey 0.20, ez 0) and u2 (ey 0.05, ez 0.35):
    chi2 = 1.04 against 0.065 + 1.42 = 1.48, the link goes to u1; with the z term subtracted it would go to u2."""
    row, pad, time = concat([_line(np.arange(20, 31)), _line(np.array([31]), dy=0.20), _line(np.array([31]), dy=0.05, dz=0.35)])
    r = oracle.track(_geom(), oracle.default_params(), row, pad, time)
    h30 = int(np.nonzero(row == 30.0)[0][0])
    assert r.up_raw[h30] == 11                                                  # u1 (index 11), not u2 (12)
    row, pad, time = concat([_line(np.arange(20, 31)), _line(np.array([31]), dy=0.20), _line(np.array([31]), dy=0.05, dz=0.10)])
    r = oracle.track(_geom(), oracle.default_params(), row, pad, time)
    assert r.up_raw[h30] == 12                                                  # control: u2 at ez 0.10 (chi2 0.18) wins


def test_P9_chi2_cut_is_strict():
    """Three hits on the pad centres of rows 29, 30, 31 (y = 0 exactly) at times 100, 101, 103: ey = 0 and ez = 2Z - Z = Z exactly,
    so chi2 = fl(fl(Z Z) w_z) -- one value, computed here from the oracle's own rounded w_z.  The link needs chi2 < chi2_cut."""
    g = _geom()
    rows = np.array([29, 30, 31])
    rowv = rows.astype(np.float32)
    padv = (0.5 * (n_pads(rows) - 1)).astype(np.float32)                       # c_r: exact in fp32
    timev = np.array([100.0, 101.0, 103.0], np.float32)
    _, _, _, consts = oracle.tables(g, oracle.default_params())
    Z = np.float32(ZBIN)
    chi2 = np.float32(np.float32(Z * Z) * np.float32(consts["wz"]))
    assert 1.0 < chi2 < 9.0
    p = oracle.default_params()
    p.chi2_cut = float(chi2)
    assert oracle.track(g, p, rowv, padv, timev).up_raw[1] == -1
    p.chi2_cut = float(np.nextafter(chi2, np.float32(100.0)))
    assert oracle.track(g, p, rowv, padv, timev).up_raw[1] == 2


def test_P10_transport_count_of_one_straight_track():
    """Row steps of a lone noise-free line on rows 20 .. 60 (statistics block of the oracle = the units of the constructor's
    roofline).  Rows 20 and 60 carry no link (a link needs both neighbours), so the start hit is row 21 and the cleaned chain
    ends on row 59:  chain 22 .. 59 = 38;  following up: row 60 (found) + 61 .. 70 (ten misses) = 11;  down pass: 60 .. 21 through
    the collected hits = 40, row 20 (found by the search) + 19 .. 10 (ten misses) = 11.  100 in all, 41 hits."""
    r, row = _track_one([_line(np.arange(20, 61))])
    assert len(r.tl_seed) == 1 and int(row[r.tl_seed[0]]) == 21 and r.tl_n_hits[0] == 41
    assert r.stats["transports"] == 100.0
    assert r.stats["updates"] == 38 + 1 + 40 + 1                                # every transport that met a hit


@pytest.mark.parametrize("n_hits,is_track", [(30, True), (29, False)])
def test_P11_a_tracklet_with_exactly_min_hits_is_a_track(n_hits, is_track):
    """B:L7 '>= 30 unshared hits': 30 hits make a track, 29 do not."""
    r, row = _track_one([_line(np.arange(20, 20 + n_hits))])
    assert len(r.tl_seed) == 1 and r.tl_n_hits[0] == n_hits
    assert len(r.tr_seed) == (1 if is_track else 0)
    if is_track:
        assert r.tr_n_hits[0] == 30


def test_P12_result_does_not_depend_on_the_input_order_with_cluster_0_in_every_role():
    """C1: 'the result is order-free (all ties break on the original cluster index)'.  The same small frame with one chosen
    cluster swapped to index 0 -- a start hit, the top hit of a tracklet, a hit in the middle of one, a hit no tracklet holds --
    must give the same links, tracklets, fits (bit for bit) and tracks once indices are mapped back."""
    tf = _small_frame(6, n_tracks=12)
    g, p = _geom(1, tf.max_time_bin), oracle.default_params(0.08, 0.12)
    base = oracle.track(g, p, tf.row, tf.pad, tf.time)
    assert len(base.tl_seed) > 20 and len(base.tr_seed) >= 8
    t_long = int(np.argmax(base.tl_n_hits))
    rows_t = np.nonzero(base.tl_row_hit[t_long] >= 0)[0]
    held = np.zeros(tf.n, bool)
    held[base.tl_row_hit[base.tl_row_hit >= 0]] = True
    roles = {"start hit": int(base.tl_seed[t_long]), "top hit": int(base.tl_row_hit[t_long, rows_t[-1]]),
             "middle hit": int(base.tl_row_hit[t_long, rows_t[len(rows_t) // 2]]), "bottom hit": int(base.tl_row_hit[t_long, rows_t[0]]),
             "free hit": int(np.nonzero(~held)[0][0])}

    def canon(r, new_of_old):
        old_of_new = np.argsort(new_of_old)
        m = lambda a: np.where(a >= 0, old_of_new[np.maximum(a, 0)], -1)
        order = np.argsort(m(r.tl_seed))
        ko = np.argsort(m(r.tr_seed))
        hits = [tuple(sorted(m(r.tr_hit_index[r.tr_hit_offset[k]:r.tr_hit_offset[k] + r.tr_n_hits[k]]))) for k in ko]
        return (m(r.link_up)[new_of_old], m(r.link_down)[new_of_old], m(r.tl_seed)[order], m(r.tl_row_hit)[order], r.tl_par[order],
                m(r.tr_seed)[ko], r.tr_par[ko], hits)

    ref = canon(base, np.arange(tf.n))
    for role, c in roles.items():
        if c == 0:
            continue
        new_of_old = np.arange(tf.n)
        new_of_old[[0, c]] = [c, 0]                                             # old cluster c sits at index 0, old cluster 0 at c
        perm = np.argsort(new_of_old)                                           # perm[new] = old
        r = oracle.track(g, p, tf.row[perm], tf.pad[perm], tf.time[perm])
        got = canon(r, new_of_old)
        for i, (a, b) in enumerate(zip(ref[:7], got[:7])):
            assert np.array_equal(a, b), (role, i)
        assert ref[7] == got[7], role
